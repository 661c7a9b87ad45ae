// inst_slab_f32.cu -- time-slab kernels (slab_kernels.cuh) for float fields, all link formats and boundary-phase kinds
#include "slab_launch.cuh"
namespace lqcd {
template lqcd_status launch_slab<float>(LQCD_LAUNCH_SLAB_ARGS);
template lqcd_status launch_push_faces<float>(LQCD_LAUNCH_FACES_ARGS);
}

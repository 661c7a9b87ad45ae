// inst_slab_f64.cu -- time-slab kernels (slab_kernels.cuh) for double fields, all link formats and boundary-phase kinds
#include "slab_launch.cuh"
namespace lqcd {
template lqcd_status launch_slab<double>(LQCD_LAUNCH_SLAB_ARGS);
template lqcd_status launch_push_faces<double>(LQCD_LAUNCH_FACES_ARGS);
}

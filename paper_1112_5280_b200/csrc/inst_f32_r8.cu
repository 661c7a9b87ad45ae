// inst_f32_r8.cu -- dslash_kernel<float, 8, ...> for all epilogues and boundary-phase kinds (launch.cuh)
#include "launch.cuh"
namespace lqcd {
template lqcd_status launch_recon<float, 8>(LQCD_LAUNCH_RECON_ARGS);
}

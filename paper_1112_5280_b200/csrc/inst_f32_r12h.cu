// inst_f32_r12h.cu -- dslash_kernel<float, RECON_12H, ...> for all epilogues and boundary-phase kinds (launch.cuh)
#include "launch.cuh"
namespace lqcd {
template lqcd_status launch_recon<float, RECON_12H>(LQCD_LAUNCH_RECON_ARGS);
}

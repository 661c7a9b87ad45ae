// inst_f32_r12.cu -- dslash_kernel<float, 12, ...> for all epilogues and boundary-phase kinds (launch.cuh)
#include "launch.cuh"
namespace lqcd {
template lqcd_status launch_recon<float, 12>(LQCD_LAUNCH_RECON_ARGS);
}

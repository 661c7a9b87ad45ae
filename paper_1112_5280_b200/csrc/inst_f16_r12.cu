// inst_f16_r12.cu -- dslash_kernel<__half, 12, ...> for all epilogues and boundary-phase kinds (launch.cuh)
#include "launch.cuh"
namespace lqcd {
template lqcd_status launch_recon<__half, 12>(LQCD_LAUNCH_RECON_ARGS);
}

// inst_f64_r12.cu -- dslash_kernel<double, 12, ...> for all epilogues and boundary-phase kinds (launch.cuh)
#include "launch.cuh"
namespace lqcd {
template lqcd_status launch_recon<double, 12>(LQCD_LAUNCH_RECON_ARGS);
}

// inst_f64_r8.cu -- dslash_kernel<double, 8, ...> for all epilogues and boundary-phase kinds (launch.cuh)
#include "launch.cuh"
namespace lqcd {
template lqcd_status launch_recon<double, 8>(LQCD_LAUNCH_RECON_ARGS);
}

// inst_f32_r18.cu -- dslash_kernel<float, 18, ...> for all epilogues and boundary-phase kinds (launch.cuh)
#include "launch.cuh"
namespace lqcd {
template lqcd_status launch_recon<float, 18>(LQCD_LAUNCH_RECON_ARGS);
}

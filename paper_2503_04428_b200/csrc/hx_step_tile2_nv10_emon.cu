// NV = 10 with the monitoring of the internal energy (Eq. 10-12): the two runtime-switch builds.
#include "hx_step_tile2_launch.cuh"
namespace hx {
namespace t2 {
cudaError_t launch_nv10_rad_emon(Plan& plan, const Args& a, int cur, cudaStream_t st);
template <>
cudaError_t launch_emon<10>(Plan& plan, const Args& a, int cur, cudaStream_t st) {
  if (a.s.P.eos == HX_EOS_GAS_RADIATION) return launch_nv10_rad_emon(plan, a, cur, st);   // own translation unit
  return launch_generic<10, true>(plan, a, cur, st);
}
}  // namespace t2
}  // namespace hx

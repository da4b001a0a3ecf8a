// NV = 6 (3-D, one passive scalar): runtime-switch build only.
#include "hx_step_tile2_launch.cuh"
namespace hx {
namespace t2 {
cudaError_t launch_nv6_rad(Plan& plan, const Args& a, int cur, cudaStream_t st);
template <>
cudaError_t launch_nv<6>(Plan& plan, const Args& a, int cur, cudaStream_t st) {
  if (a.s.P.emon_eps > 0.0) return launch_emon<6>(plan, a, cur, st);   // Eq. 10-12 (ideal gas; checked by tile2_supported): own translation unit
  if (a.s.P.eos == HX_EOS_GAS_RADIATION) return launch_nv6_rad(plan, a, cur, st);   // Eq. 6-7: own translation unit
  return launch_generic<6>(plan, a, cur, st);
}
}  // namespace t2
}  // namespace hx

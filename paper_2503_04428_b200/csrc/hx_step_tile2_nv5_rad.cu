// NV = 5 with the gas + radiation EOS (Eq. 6-7): the two runtime-switch builds.  Own translation unit (compile time).
#include "hx_step_tile2_launch.cuh"
namespace hx {
namespace t2 {
cudaError_t launch_nv5_rad(Plan& plan, const Args& a, int cur, cudaStream_t st) {
  const Phys& P = a.s.P;
  if (P.spherical) return launch_cfg<5, true, GRAV_ANY, -1, -1, false, HX_EOS_GAS_RADIATION>(plan, a, cur, st);
  return launch_cfg<5, false, GRAV_ANY, -1, -1, false, HX_EOS_GAS_RADIATION>(plan, a, cur, st);
}
}  // namespace t2
}  // namespace hx

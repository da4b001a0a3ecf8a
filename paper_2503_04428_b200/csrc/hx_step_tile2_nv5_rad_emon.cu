// NV = 5 with the gas + radiation EOS (Eq. 6-7) AND the monitoring of the internal energy (Eq. 10-12) -- the combination of the
// paper's supernova runs (L377, L120-L126): the two runtime-switch builds.  Own translation unit (compile time).
#include "hx_step_tile2_launch.cuh"
namespace hx {
namespace t2 {
cudaError_t launch_nv5_rad_emon(Plan& plan, const Args& a, int cur, cudaStream_t st) {
  if (a.s.P.spherical) return launch_cfg<5, true, GRAV_ANY, -1, -1, false, HX_EOS_GAS_RADIATION, true>(plan, a, cur, st);
  return launch_cfg<5, false, GRAV_ANY, -1, -1, false, HX_EOS_GAS_RADIATION, true>(plan, a, cur, st);
}
}  // namespace t2
}  // namespace hx

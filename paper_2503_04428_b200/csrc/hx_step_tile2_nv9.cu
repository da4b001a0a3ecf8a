// NV = 9 (3-D, four passive scalars).  Fully specialised: spherical wedge with point-mass gravity, minmod + HLLC
// (config 5, wedge_3d).
#include "hx_step_tile2_launch.cuh"
namespace hx {
namespace t2 {
cudaError_t launch_nv9_rad(Plan& plan, const Args& a, int cur, cudaStream_t st);
template <>
cudaError_t launch_nv<9>(Plan& plan, const Args& a, int cur, cudaStream_t st) {
  if (a.s.P.emon_eps > 0.0) return launch_emon<9>(plan, a, cur, st);   // Eq. 10-12 (ideal gas; checked by tile2_supported): own translation unit
  const Phys& P = a.s.P;
  if (P.eos == HX_EOS_GAS_RADIATION) return launch_nv9_rad(plan, a, cur, st);   // Eq. 6-7: own translation unit (compile time)
  if (P.spherical && plan.grav_r && P.limiter == HX_LIM_MINMOD && P.riemann == HX_RIEMANN_HLLC)
    return launch_cfg<9, true, GRAV_R, HX_LIM_MINMOD, HX_RIEMANN_HLLC, false>(plan, a, cur, st);
  return launch_generic<9>(plan, a, cur, st);
}
}  // namespace t2
}  // namespace hx

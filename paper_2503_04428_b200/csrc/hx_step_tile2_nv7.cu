// NV = 7 (3-D, two passive scalars).  Fully specialised: Cartesian, gravity along z, MC + HLLC (config 4, rt_3d).
#include "hx_step_tile2_launch.cuh"
namespace hx {
namespace t2 {
cudaError_t launch_nv7_rad(Plan& plan, const Args& a, int cur, cudaStream_t st);
template <>
cudaError_t launch_nv<7>(Plan& plan, const Args& a, int cur, cudaStream_t st) {
  if (a.s.P.emon_eps > 0.0) return launch_emon<7>(plan, a, cur, st);   // Eq. 10-12 (ideal gas; checked by tile2_supported): own translation unit
  if (a.s.P.eos == HX_EOS_GAS_RADIATION) return launch_nv7_rad(plan, a, cur, st);   // Eq. 6-7: own translation unit
  const Phys& P = a.s.P;
  if (!P.spherical && plan.grav_z && P.limiter == HX_LIM_MC && P.riemann == HX_RIEMANN_HLLC) {
    if (plan.uni) return launch_cfg<7, false, GRAV_Z, HX_LIM_MC, HX_RIEMANN_HLLC, true>(plan, a, cur, st);
    return launch_cfg<7, false, GRAV_Z, HX_LIM_MC, HX_RIEMANN_HLLC, false>(plan, a, cur, st);
  }
  return launch_generic<7>(plan, a, cur, st);
}
}  // namespace t2
}  // namespace hx

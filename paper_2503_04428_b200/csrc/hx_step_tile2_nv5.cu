// NV = 5 (3-D, no passive scalar).  Fully specialised: no gravity, minmod + HLLC, Cartesian (config 3, sedov_3d) and
// spherical (the paper's off-centre Sedov wedge, Sect. 4.3).
#include "hx_step_tile2_launch.cuh"
namespace hx {
namespace t2 {
cudaError_t launch_nv5_rad(Plan& plan, const Args& a, int cur, cudaStream_t st);
template <>
cudaError_t launch_nv<5>(Plan& plan, const Args& a, int cur, cudaStream_t st) {
  if (a.s.P.emon_eps > 0.0) return launch_emon<5>(plan, a, cur, st);   // Eq. 10-12 (ideal gas; checked by tile2_supported): own translation unit
  if (a.s.P.eos == HX_EOS_GAS_RADIATION) return launch_nv5_rad(plan, a, cur, st);   // Eq. 6-7: own translation unit
  const Phys& P = a.s.P;
  if (!P.spherical && P.gravity == HX_GRAV_NONE && P.limiter == HX_LIM_MINMOD && P.riemann == HX_RIEMANN_HLLC) {
    if (plan.uni && plan.ty == 12) return launch_cfg<5, false, GRAV_OFF, HX_LIM_MINMOD, HX_RIEMANN_HLLC, true, HX_EOS_IDEAL, false, 12>(plan, a, cur, st);
    if (plan.uni) return launch_cfg<5, false, GRAV_OFF, HX_LIM_MINMOD, HX_RIEMANN_HLLC, true>(plan, a, cur, st);
    return launch_cfg<5, false, GRAV_OFF, HX_LIM_MINMOD, HX_RIEMANN_HLLC, false>(plan, a, cur, st);
  }
  if (P.spherical && P.gravity == HX_GRAV_NONE && P.limiter == HX_LIM_MINMOD && P.riemann == HX_RIEMANN_HLLC)
    return launch_cfg<5, true, GRAV_OFF, HX_LIM_MINMOD, HX_RIEMANN_HLLC, false>(plan, a, cur, st);
  return launch_generic<5>(plan, a, cur, st);
}
}  // namespace t2
}  // namespace hx

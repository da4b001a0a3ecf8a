// NV = 10 (3-D, five passive scalars: the field count of the paper's supernova runs, Sect. 5.5).  Fully specialised: spherical, minmod + HLLC; runtime-switch builds for the rest.
#include "hx_step_tile2_launch.cuh"
namespace hx {
namespace t2 {
cudaError_t launch_nv10_rad(Plan& plan, const Args& a, int cur, cudaStream_t st);
template <>
cudaError_t launch_nv<10>(Plan& plan, const Args& a, int cur, cudaStream_t st) {
  if (a.s.P.emon_eps > 0.0) return launch_emon<10>(plan, a, cur, st);   // Eq. 10-12 (ideal gas; checked by tile2_supported): own translation unit
  const Phys& P = a.s.P;
  if (P.eos == HX_EOS_GAS_RADIATION) return launch_nv10_rad(plan, a, cur, st);
  if (P.spherical && plan.grav_r && P.limiter == HX_LIM_MINMOD && P.riemann == HX_RIEMANN_HLLC)
    return launch_cfg<10, true, GRAV_R, HX_LIM_MINMOD, HX_RIEMANN_HLLC, false>(plan, a, cur, st);
  return launch_generic<10>(plan, a, cur, st);
}
}  // namespace t2
}  // namespace hx

// NV = 5 with the monitoring of the internal energy (Eq. 10-12): the cold_stream_3d build and the two runtime-switch builds.
#include "hx_step_tile2_launch.cuh"
namespace hx {
namespace t2 {
cudaError_t launch_nv5_rad_emon(Plan& plan, const Args& a, int cur, cudaStream_t st);
template <>
cudaError_t launch_emon<5>(Plan& plan, const Args& a, int cur, cudaStream_t st) {
  if (a.s.P.eos == HX_EOS_GAS_RADIATION) return launch_nv5_rad_emon(plan, a, cur, st);   // own translation unit
  const Phys& P = a.s.P;
  // fully specialised: Cartesian, no gravity, MC + HLLC (cold_stream_3d)
  if (!P.spherical && P.gravity == HX_GRAV_NONE && P.limiter == HX_LIM_MC && P.riemann == HX_RIEMANN_HLLC) {
    if (plan.uni) return launch_cfg<5, false, GRAV_OFF, HX_LIM_MC, HX_RIEMANN_HLLC, true, HX_EOS_IDEAL, true>(plan, a, cur, st);
    return launch_cfg<5, false, GRAV_OFF, HX_LIM_MC, HX_RIEMANN_HLLC, false, HX_EOS_IDEAL, true>(plan, a, cur, st);
  }
  return launch_generic<5, true>(plan, a, cur, st);
}
}  // namespace t2
}  // namespace hx

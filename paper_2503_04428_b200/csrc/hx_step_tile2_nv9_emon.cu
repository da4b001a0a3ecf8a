// NV = 9 with the monitoring of the internal energy (Eq. 10-12): the spherical wedge build (wedge_3d_emon) and the two runtime-switch builds.
#include "hx_step_tile2_launch.cuh"
namespace hx {
namespace t2 {
cudaError_t launch_nv9_rad_emon(Plan& plan, const Args& a, int cur, cudaStream_t st);
template <>
cudaError_t launch_emon<9>(Plan& plan, const Args& a, int cur, cudaStream_t st) {
  if (a.s.P.eos == HX_EOS_GAS_RADIATION) return launch_nv9_rad_emon(plan, a, cur, st);   // own translation unit
  const Phys& P = a.s.P;
  // fully specialised: spherical wedge, radial gravity, minmod + HLLC (wedge_3d_emon: the paper's use case, highly supersonic ejecta, L120-L126)
  if (P.spherical && plan.grav_r && P.limiter == HX_LIM_MINMOD && P.riemann == HX_RIEMANN_HLLC)
    return launch_cfg<9, true, GRAV_R, HX_LIM_MINMOD, HX_RIEMANN_HLLC, false, HX_EOS_IDEAL, true>(plan, a, cur, st);
  return launch_generic<9, true>(plan, a, cur, st);
}
}  // namespace t2
}  // namespace hx

// NV = 9 with the gas + radiation EOS (Eq. 6-7) AND the monitoring of the internal energy (Eq. 10-12) -- the combination of the
// paper's supernova runs (L377, L120-L126): the spherical radial-gravity minmod + HLLC build and the two runtime-switch builds.  Own translation unit (compile time).
#include "hx_step_tile2_launch.cuh"
namespace hx {
namespace t2 {
cudaError_t launch_nv9_rad_emon(Plan& plan, const Args& a, int cur, cudaStream_t st) {
  const Phys& P = a.s.P;
  // fully specialised: spherical wedge, radial gravity, minmod + HLLC (wedge_3d_sn_emon: the paper's supernova setup with everything on)
  if (P.spherical && plan.grav_r && P.limiter == HX_LIM_MINMOD && P.riemann == HX_RIEMANN_HLLC)
    return launch_cfg<9, true, GRAV_R, HX_LIM_MINMOD, HX_RIEMANN_HLLC, false, HX_EOS_GAS_RADIATION, true>(plan, a, cur, st);
  if (a.s.P.spherical) return launch_cfg<9, true, GRAV_ANY, -1, -1, false, HX_EOS_GAS_RADIATION, true>(plan, a, cur, st);
  return launch_cfg<9, false, GRAV_ANY, -1, -1, false, HX_EOS_GAS_RADIATION, true>(plan, a, cur, st);
}
}  // namespace t2
}  // namespace hx

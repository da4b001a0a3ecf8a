// hx_step_tile2_launch.cuh -- launch dispatch of the fused step kernel for one field count NV.  Each
// hx_step_tile2_nv<N>.cu instantiates launch_nv<N> so the variants compile in parallel.
#pragma once
#include "hx_step_tile2.cuh"

namespace hx {
namespace t2 {

struct Plan {
  CUtensorMap tmap[2];
  int ndim;          // 3: hx_step_tile2.cuh (march along z); 2: hx_step_tile2d.cuh (march along y)
  int zc;            // planes (rows in 2-D) per chunk of the march direction
  int ty;            // owner rows of a 3-D tile: 8, or 12 for the configuration tile_rows() names
  int bcx_lo, bcx_hi; // boundary conditions of direction 0 (some 3-D builds write the x-ghost cells themselves)
  bool xghost;       // the build launched last wrote the x-ghost cells of the interior rows (set by launch_cfg)
  dim3 grid;
  bool uni;          // bitwise-uniform Cartesian tables: geometry travels as kernel-parameter constants
  bool grav_z;       // uniform gravity along direction 2 only
  bool grav_r;       // spherical point mass / self-gravity: acceleration along direction 0 only
  double uf[3], uiw[3];
  const char* name;
};

template <int NV>
cudaError_t launch_nv(Plan& plan, const Args& a, int cur, cudaStream_t st);

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute of a kernel: raise it (never lower it) once per
// (kernel, device), under a lock -- handles of one process may live on several GPUs and step from several threads.
cudaError_t set_smem_limit(const void* kern, size_t smem);

// Owner rows per tile.  Twelve rows (three owner warps + one ring warp per scheduler, 136 registers per owner thread) carry less
// ring work per cell; they pay only where the owner path fits into those registers: nvar 5, Cartesian, constant geometry, no
// gravity, minmod + HLLC (config 3: sedov_3d 0.970 -> 0.936 ms; nvar 7 spills and needs two z chunks: 10.30 -> 12.69 ms;
// the spherical nvar-5 build: 1.11 -> 1.22 ms).  One place decides, for the plan (grid, shared memory) and for the dispatch.
inline int tile_rows(const Layout& L, const Phys& P, bool uni) {
  const bool c3 = L.nvar == 5 && !P.spherical && uni && P.gravity == HX_GRAV_NONE && P.limiter == HX_LIM_MINMOD && P.riemann == HX_RIEMANN_HLLC &&
                  P.eos == HX_EOS_IDEAL && !(P.emon_eps > 0.0) && L.n[1] >= 24 &&
                  ((L.n[1] + 11) / 12 * 12 - L.n[1]) * 25 <= L.n[1];   // at most 4 % of the tile rows beyond the grid
  return c3 ? 12 : TY_DEFAULT;
}

template <int NV, bool SPH, int GRAV, int LIM, int RS, bool UNI, int EOS = HX_EOS_IDEAL, bool EMON = false, int TY = TY_DEFAULT>
static cudaError_t launch_cfg(Plan& plan, const Args& a_in, int cur, cudaStream_t st) {
  if (plan.ty != TY) return cudaErrorInvalidConfiguration;   // the plan's grid and shared memory were sized for another tile height
  Args a = a_in;
  if (UNI && LIM == HX_LIM_MC)   // a build with a static limiter folds its lim_scale (1/2 for MC) into the uniform slope pre-scale
    for (int d = 0; d < 3; ++d) a.uf[d] *= 0.5;
  auto kern = step_tile2_kernel<NV, SPH, GRAV, LIM, RS, UNI, TY, EOS, EMON>;
  const size_t smem = Smem<NV, TY>::total(plan.zc, SPH);
  cudaError_t e = set_smem_limit((const void*)kern, smem);
  if (e != cudaSuccess) return e;
  plan.xghost = writes_x_ghosts(UNI, TY);
  plan.name = EMON ? (EOS != HX_EOS_IDEAL ? "tile2_rad_emon" : (UNI ? "tile2_emon_uni" : "tile2_emon")) : (UNI ? (TY == 12 ? "tile2_uni12" : "tile2_uni") : (EOS == HX_EOS_IDEAL ? "tile2" : "tile2_rad"));
  kern<<<plan.grid, (TY + 4) * 32, smem, st>>>(plan.tmap[cur], a);
  return cudaGetLastError();
}

// the runtime-switch build (limiter, solver, any gravity) covers every configuration of this NV
template <int NV, bool EMON = false>
static cudaError_t launch_generic(Plan& plan, const Args& a, int cur, cudaStream_t st) {
  if (a.s.P.spherical) return launch_cfg<NV, true, GRAV_ANY, -1, -1, false, HX_EOS_IDEAL, EMON>(plan, a, cur, st);
  if (plan.uni && !EMON) return launch_cfg<NV, false, GRAV_ANY, -1, -1, true, HX_EOS_IDEAL, EMON>(plan, a, cur, st);   // bitwise-uniform Cartesian grid
  return launch_cfg<NV, false, GRAV_ANY, -1, -1, false, HX_EOS_IDEAL, EMON>(plan, a, cur, st);
}

// internal-energy monitoring (Eq. 10-12), ideal gas: one translation unit per NV (hx_step_tile2_nv<N>_emon.cu)
template <int NV>
cudaError_t launch_emon(Plan& plan, const Args& a, int cur, cudaStream_t st);

}  // namespace t2
}  // namespace hx

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

template <int NV, bool SPH, int GRAV, int LIM, int RS, bool UNI, int EOS = HX_EOS_IDEAL, bool EMON = false>
static cudaError_t launch_cfg(Plan& plan, const Args& a_in, int cur, cudaStream_t st) {
  constexpr int TY = TY_DEFAULT;
  Args a = a_in;
  if (UNI && LIM == HX_LIM_MC)   // a build with a static limiter folds its lim_scale (1/2 for MC) into the uniform slope pre-scale
    for (int d = 0; d < 3; ++d) a.uf[d] *= 0.5;
  auto kern = step_tile2_kernel<NV, SPH, GRAV, LIM, RS, UNI, TY, EOS, EMON>;
  const size_t smem = Smem<NV, TY>::total(plan.zc, SPH);
  cudaError_t e = set_smem_limit((const void*)kern, smem);
  if (e != cudaSuccess) return e;
  plan.name = EMON ? (UNI ? "tile2_emon_uni" : "tile2_emon") : (UNI ? "tile2_uni" : (EOS == HX_EOS_IDEAL ? "tile2" : "tile2_rad"));
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

// hx_step_tile2d.cu -- host side of the fused 2-D step kernel (hx_step_tile2d.cuh): tensor maps over the padded SoA
// state (x, y, field), launch geometry, dispatch on the field count and on the specialised configurations.
#include "hx_step_tile2_launch.cuh"
#include "hx_step_tile2d.cuh"

namespace hx {

using t2::Plan;

static size_t smem_fixed_2d(int nv) {
  switch (nv) {
    case 4: return t2d::Smem<4>::fixed;
    case 5: return t2d::Smem<5>::fixed;
    case 6: return t2d::Smem<6>::fixed;
    case 7: return t2d::Smem<7>::fixed;
    case 8: return t2d::Smem<8>::fixed;
    default: return 0;
  }
}

// Cartesian 2-D grids, ideal gas, no internal-energy monitoring, nvar 4..8 (up to four passive scalars), no gravity or
// uniform gravity; everything else in 2-D runs on the generic kernel.
int tile2d_supported(const Layout& L, const Phys& P) {
  return L.ndim == 2 && !P.spherical && P.eos == HX_EOS_IDEAL && !(P.emon_eps > 0.0) && L.nvar >= 4 && L.nvar <= 8 &&
         (P.gravity == HX_GRAV_NONE || P.gravity == HX_GRAV_UNIFORM) && L.n[0] >= 2 && L.n[1] >= 2;
}

// Fill the launch geometry and the two tensor maps of a 2-D plan.  `enc` is cuTensorMapEncodeTiled.
cudaError_t tile2d_plan_fill(Plan* p, const Layout& L, double* const U[2], const double* uni, void* enc_fn) {
  typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                    const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  EncodeTiledFn enc = (EncodeTiledFn)enc_fn;
  int sms = 148;
  {
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaGetDeviceProperties(&prop, dev) == cudaSuccess && prop.multiProcessorCount > 0)
      sms = prop.multiProcessorCount;
  }
  const int ntx = (L.n[0] + t2d::TXS - 1) / t2d::TXS;
  // y chunks: every chunk marches 3 extra rows (+ a prologue); one CTA per SM at a time, waves of `sms` CTAs: pick the
  // chunk count that maximises (useful rows / rows marched) x (waves / whole waves); at least 8 rows per chunk
  const size_t fixed = smem_fixed_2d(L.nvar), budget = 227 * 1024 - 1024;
  int best_chunks = 1;
  double best = -1.0;
  for (int c = 1; c <= (L.n[1] + 7) / 8; ++c) {
    const int yc = (L.n[1] + c - 1) / c, chunks = (L.n[1] + yc - 1) / yc;
    if (fixed + 5 * (size_t)(yc + 6) * 8 > budget) continue;
    const double waves = (double)((long long)ntx * chunks) / sms;
    const double eff = (double)L.n[1] / ((double)chunks * (yc + 4)) * waves / (double)(long long)(waves + 0.999999);
    if (eff > best + 1e-9) {
      best = eff;
      best_chunks = chunks;
    }
  }
  p->zc = (L.n[1] + best_chunks - 1) / best_chunks;
  const int nyc = (L.n[1] + p->zc - 1) / p->zc;
  p->grid = dim3((unsigned)ntx, (unsigned)nyc, 1u);
  p->ndim = 2;
  p->ty = 0;
  p->uni = uni != nullptr;
  p->grav_z = false;
  p->grav_r = false;
  for (int d = 0; d < 3; ++d) {
    p->uf[d] = uni ? uni[d] : 0.0;
    p->uiw[d] = uni ? uni[3 + d] : 0.0;
  }
  p->name = "tile2d";
  for (int b = 0; b < 2; ++b) {
    const cuuint64_t dims[3] = {(cuuint64_t)L.sy, (cuuint64_t)L.np[1], (cuuint64_t)L.nvar};
    const cuuint64_t strides[2] = {(cuuint64_t)L.sy * 8, (cuuint64_t)L.sv * 8};
    const cuuint32_t box[3] = {(cuuint32_t)t2d::HXS, 1u, (cuuint32_t)L.nvar};   // half a staged row (a box is at most 256 wide)
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    CUresult r = enc(&p->tmap[b], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void*)U[b], dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
  }
  return cudaSuccess;
}

namespace t2d {

template <int NV, int GRAV, int LIM, int RS, bool UNI>
static cudaError_t launch_cfg(Plan& plan, const Args& a_in, int cur, cudaStream_t st) {
  auto kern = step_tile2d_kernel<NV, GRAV, LIM, RS, UNI>;
  Args a = a_in;
  if (UNI && LIM == HX_LIM_MC)   // a build with a static limiter folds its lim_scale (1/2 for MC) into the uniform slope pre-scale
    for (int d = 0; d < 2; ++d) a.uf[d] *= 0.5;
  const size_t smem = Smem<NV>::total(plan.zc);
  cudaError_t e = t2::set_smem_limit((const void*)kern, smem);
  if (e != cudaSuccess) return e;
  plan.name = UNI ? "tile2d_uni" : "tile2d";
  kern<<<plan.grid, NTHREADS, smem, st>>>(plan.tmap[cur], a);
  return cudaGetLastError();
}

template <int NV>
static cudaError_t launch_nv(Plan& plan, const Args& a, int cur, cudaStream_t st) {
  const Phys& P = a.s.P;
  // fully specialised: bitwise-uniform grid, no gravity, HLLC with MC (config 2, kh_2d) or minmod
  if (plan.uni && P.gravity == HX_GRAV_NONE && P.riemann == HX_RIEMANN_HLLC) {
    if (P.limiter == HX_LIM_MC) return launch_cfg<NV, GRAV_OFF, HX_LIM_MC, HX_RIEMANN_HLLC, true>(plan, a, cur, st);
    if (P.limiter == HX_LIM_MINMOD) return launch_cfg<NV, GRAV_OFF, HX_LIM_MINMOD, HX_RIEMANN_HLLC, true>(plan, a, cur, st);
  }
  if (plan.uni) return launch_cfg<NV, GRAV_ANY, -1, -1, true>(plan, a, cur, st);   // runtime switch (limiter, solver, gravity) on a bitwise-uniform grid
  return launch_cfg<NV, GRAV_ANY, -1, -1, false>(plan, a, cur, st);   // ... on any Cartesian grid
}

}  // namespace t2d

cudaError_t launch_step_tile2d(Plan* plan, const StepArgs& s, int cur, cudaStream_t st) {
  t2d::Args a;
  a.s = s;
  a.yc = plan->zc;
  const double hdt = 0.5 * s.dt;
  for (int d = 0; d < 2; ++d) {
    a.uf[d] = plan->uf[d];                                             // (launch_cfg folds in the lim_scale of a static limiter)
    a.uhc[d] = hdt * plan->uiw[d];
    a.uil[d] = plan->uiw[d];
  }
  switch (s.L.nvar) {
    case 4: return t2d::launch_nv<4>(*plan, a, cur, st);
    case 5: return t2d::launch_nv<5>(*plan, a, cur, st);
    case 6: return t2d::launch_nv<6>(*plan, a, cur, st);
    case 7: return t2d::launch_nv<7>(*plan, a, cur, st);
    case 8: return t2d::launch_nv<8>(*plan, a, cur, st);
    default: return cudaErrorNotSupported;
  }
}

}  // namespace hx

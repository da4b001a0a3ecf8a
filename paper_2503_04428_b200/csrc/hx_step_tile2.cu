// hx_step_tile2.cu -- host side of the fused 3-D step kernel (hx_step_tile2.cuh): tensor maps over the
// padded SoA state, launch geometry, uniform-grid detection, dispatch on the field count.
#include <cstring>
#include <map>
#include <mutex>
#include <utility>

#include "hx_step_tile2_launch.cuh"

namespace hx {

using t2::Plan;

// 2-D kernel (hx_step_tile2d.cu)
int tile2d_supported(const Layout& L, const Phys& P);
cudaError_t tile2d_plan_fill(Plan* p, const Layout& L, double* const U[2], const double* uni, void* enc_fn);
cudaError_t launch_step_tile2d(Plan* plan, const StepArgs& s, int cur, cudaStream_t st);

cudaError_t t2::set_smem_limit(const void* kern, size_t smem) {
  static std::mutex mu;
  static std::map<std::pair<const void*, int>, size_t> done;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lock(mu);
  size_t& have = done[std::make_pair(kern, dev)];
  if (have < smem) {
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    have = smem;
  }
  return cudaSuccess;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

static size_t smem_fixed(int nv, int ty) {   // shared memory of one CTA without the z tables of its chunk
  constexpr int TY = t2::TY_DEFAULT;
  if (ty == 12) return nv == 5 ? t2::Smem<5, 12>::fixed : 0;
  switch (nv) {
    case 5: return t2::Smem<5, TY>::fixed;
    case 6: return t2::Smem<6, TY>::fixed;
    case 7: return t2::Smem<7, TY>::fixed;
    case 8: return t2::Smem<8, TY>::fixed;
    case 9: return t2::Smem<9, TY>::fixed;
    case 10: return t2::Smem<10, TY>::fixed;
    case 11: return t2::Smem<11, TY>::fixed;
    default: return 0;
  }
}

// 3-D field counts with an instantiation: up to six passive scalars (nvar 11 is the largest whose planes, exchange
// slots and private scalar slots fit into the 227 KB of shared memory a CTA can have)
static bool nv_supported(int nv) { return nv >= 5 && nv <= 11; }

int tile2_supported(const Layout& L, const Phys& P) {
  if (L.ndim == 2) return tile2d_supported(L, P);
  if (P.spherical && P.gravity == HX_GRAV_UNIFORM) return 0;   // a constant (r, theta, phi) acceleration vector: generic kernel (the spherical tile builds carry no phi gravity)
  return L.ndim == 3 && nv_supported(L.nvar) && L.n[0] >= 2 && L.n[1] >= 2 && L.n[2] >= 2;
}

// uni: non-null when every per-axis table of this Cartesian grid is bitwise constant; then uni[0..2] = hw*idx and
// uni[3..5] = 1/delta of the three axes.
int tile2_writes_x_ghosts(const Plan* p) { return p && p->ndim == 3 && p->xghost; }   // valid after a launch

cudaError_t tile2_plan_create(const Layout& L, const Phys& P, double* const U[2], const double* uni, int grav_z, int bcx_lo, int bcx_hi, Plan** out) {
  *out = nullptr;
  EncodeTiledFn enc = get_encode_fn();
  if (!enc) return cudaErrorNotSupported;
  Plan* p = new Plan();
  p->xghost = false;
  p->bcx_lo = bcx_lo;
  p->bcx_hi = bcx_hi;
  if (L.ndim == 2) {
    cudaError_t e2 = tile2d_plan_fill(p, L, U, uni, (void*)enc);
    if (e2 != cudaSuccess) {
      delete p;
      return e2;
    }
    *out = p;
    return cudaSuccess;
  }
  p->ndim = 3;
  const int TY = t2::tile_rows(L, P, uni != nullptr);
  p->ty = TY;
  const int ntx = (L.n[0] + t2::TX - 1) / t2::TX, nty = (L.n[1] + TY - 1) / TY;
  // z chunks: every chunk re-reads 4 planes and recomputes 2 predictor planes (+ a prologue), and with one CTA per
  // SM the grid runs in waves of `sms` CTAs of equal length: pick the chunk count that maximises
  // (useful planes / planes marched) x (waves / whole waves).
  int sms = 148;
  {
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaGetDeviceProperties(&prop, dev) == cudaSuccess && prop.multiProcessorCount > 0)
      sms = prop.multiProcessorCount;
  }
  const long long cols = (long long)ntx * nty;
  // the chunk's z tables live in shared memory next to the plane ring and the exchange buffers (227 KB per CTA)
  constexpr int TYs = t2::TY_DEFAULT;
  const size_t fixed = smem_fixed(L.nvar, TY) + (P.spherical ? (size_t)t2::Smem<5, TYs>::GT_N * 8 : 0);   // (GT_N does not depend on the field count)
  const size_t var_per_plane = (size_t)t2::Smem<5, TYs>::nzt(P.spherical != 0) * 8;
  const size_t budget = 227 * 1024 - 256;    // 256 B of static shared memory: the block reduction of the CFL rate
  int nzc = (L.n[2] + 15) / 16;
  double best = -1.0;
  for (int c = 1; c <= (L.n[2] + 15) / 16; ++c) {
    const int zc = (L.n[2] + c - 1) / c, chunks = (L.n[2] + zc - 1) / zc;
    if (fixed + var_per_plane * (size_t)(zc + 6) > budget) continue;
    const double waves = (double)(cols * chunks) / sms;
    const double eff = (double)L.n[2] / ((double)chunks * (zc + 3)) * waves / (double)(long long)(waves + 0.999999);
    if (eff > best + 1e-9) {
      best = eff;
      nzc = chunks;
    }
  }
  p->zc = (L.n[2] + nzc - 1) / nzc;
  nzc = (L.n[2] + p->zc - 1) / p->zc;
  p->grid = dim3((unsigned)ntx, (unsigned)nty, (unsigned)nzc);
  p->uni = uni != nullptr;
  p->grav_z = grav_z != 0;
  p->grav_r = P.spherical && (P.gravity == HX_GRAV_POINT_MASS || P.gravity == HX_GRAV_SELF);
  for (int d = 0; d < 3; ++d) {
    p->uf[d] = uni ? uni[d] : 0.0;
    p->uiw[d] = uni ? uni[3 + d] : 0.0;
  }
  p->name = "tile2";
  for (int b = 0; b < 2; ++b) {
    const cuuint64_t dims[4] = {(cuuint64_t)L.sy, (cuuint64_t)L.np[1], (cuuint64_t)L.np[2], (cuuint64_t)L.nvar};
    const cuuint64_t strides[3] = {(cuuint64_t)L.sy * 8, (cuuint64_t)L.sz * 8, (cuuint64_t)L.sv * 8};
    const cuuint32_t box[4] = {(cuuint32_t)t2::PX, (cuuint32_t)(TY + 4), 1u, (cuuint32_t)L.nvar};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    CUresult r = enc(&p->tmap[b], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void*)U[b], dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
      delete p;
      return cudaErrorInvalidValue;
    }
  }
  *out = p;
  return cudaSuccess;
}

void tile2_plan_destroy(Plan* p) { delete p; }
const char* tile2_kernel_name(const Plan* p) { return p ? p->name : "tile2"; }

cudaError_t launch_step_tile2(Plan* plan, const StepArgs& s, int cur, cudaStream_t st) {
  if (plan->ndim == 2) return launch_step_tile2d(plan, s, cur, st);
  t2::Args a;
  a.s = s;
  a.zc = plan->zc;
  a.bcx_lo = plan->bcx_lo;
  a.bcx_hi = plan->bcx_hi;
  const double hdt = 0.5 * s.dt;
  for (int d = 0; d < 3; ++d) {
    a.uf[d] = plan->uf[d];                                             // (launch_cfg folds in the lim_scale of a static limiter)
    a.uhc[d] = hdt * plan->uiw[d];
    a.uil[d] = plan->uiw[d];
  }
  switch (s.L.nvar) {
    case 5: return t2::launch_nv<5>(*plan, a, cur, st);
    case 6: return t2::launch_nv<6>(*plan, a, cur, st);
    case 7: return t2::launch_nv<7>(*plan, a, cur, st);
    case 8: return t2::launch_nv<8>(*plan, a, cur, st);
    case 9: return t2::launch_nv<9>(*plan, a, cur, st);
    case 10: return t2::launch_nv<10>(*plan, a, cur, st);
    case 11: return t2::launch_nv<11>(*plan, a, cur, st);
    default: return cudaErrorNotSupported;
  }
}

}  // namespace hx

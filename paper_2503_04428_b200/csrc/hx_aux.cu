// hx_aux.cu -- ghost / boundary fill (A0), pack / unpack between the caller's interior buffer and
// the padded arrays (with optional prim <-> cons through the EOS), stand-alone CFL reduction (A7).
// PAPER.md L203 (boundary conditions), Eq. 5 (EOS), R2 (CFL), R16-R17 (ghost layers).
#include "hx_common.cuh"

namespace hx {

// One direction of the ordered ghost fill.  Work item = (field, transverse cell, side, layer).
// Transverse extent: full padded range for directions already filled (e < d), interior range
// for directions still to come (e > d) -- identical result to sweeping the full padded extent
// because later passes overwrite those cells anyway.
__global__ void ghost_fill_kernel(Layout L, double* __restrict__ U, int d, int bc_lo, int bc_hi) {
  int ext[3], base[3];
  for (int e = 0; e < 3; ++e) {
    if (e < d) { ext[e] = L.np[e]; base[e] = 0; }
    else { ext[e] = L.n[e]; base[e] = L.ng[e]; }
  }
  ext[d] = 2 * NG;   // side * NG + layer
  const long long per_field = (long long)ext[0] * ext[1] * ext[2];
  const long long total = per_field * L.nvar;
  const int n = L.n[d];
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
    const int v = (int)(t / per_field);
    long long r = t % per_field;
    int c[3];
    c[0] = (int)(r % ext[0]); r /= ext[0];
    c[1] = (int)(r % ext[1]); r /= ext[1];
    c[2] = (int)r;
    const int side = c[d] / NG, g = c[d] % NG + 1;   // g = 1, 2: distance from the boundary face
    const int bc = side ? bc_hi : bc_lo;
    int src, dst;
    if (side == 0) {
      dst = -g;
      src = (bc == HX_BC_PERIODIC) ? n - g : (bc == HX_BC_TRANSMISSIVE ? 0 : g - 1);
    } else {
      dst = n - 1 + g;
      src = (bc == HX_BC_PERIODIC) ? g - 1 : (bc == HX_BC_TRANSMISSIVE ? n - 1 : n - g);
    }
    int p[3] = {c[0] + base[0], c[1] + base[1], c[2] + base[2]};
    p[d] = src + NG;
    double val = U[v * L.sv + L.off(p[0], p[1], p[2])];
    if ((bc == HX_BC_REFLECTING || bc == HX_BC_WEDGE) && v == 1 + d) val = -val;
    p[d] = dst + NG;
    U[v * L.sv + L.off(p[0], p[1], p[2])] = val;
  }
}

cudaError_t launch_ghost_fill(const Layout& L, double* U, int d, int bc_lo, int bc_hi, cudaStream_t s) {
  long long total = (long long)L.nvar * 2 * NG;
  for (int e = 0; e < 3; ++e)
    if (e != d) total *= (e < d) ? L.np[e] : L.n[e];
  const int block = 256;
  long long grid = (total + block - 1) / block;
  if (grid > 148LL * 16) grid = 148LL * 16;
  ghost_fill_kernel<<<(unsigned)grid, block, 0, s>>>(L, U, d, bc_lo, bc_hi);
  return cudaGetLastError();
}

// interior SoA [nvar][n2][n1][n0] (caller layout)  ->  padded state; to_cons: input is primitive
template <int ND>
__global__ void pack_kernel(Layout L, Phys P, const double* __restrict__ src, double* __restrict__ U, int to_cons) {
  const long long ncell = (long long)L.n[0] * L.n[1] * L.n[2];
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < ncell; t += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(t % L.n[0]);
    const int j = (int)((t / L.n[0]) % L.n[1]);
    const int k = (int)(t / ((long long)L.n[0] * L.n[1]));
    const long long o = L.off(i + L.ng[0], j + L.ng[1], k + L.ng[2]);
    double a[NVMAX], b[NVMAX];
    for (int v = 0; v < L.nvar; ++v) a[v] = src[v * ncell + t];
    if (to_cons) {
      prim_to_cons<ND>(P, L.nvar, a, b);
      for (int v = 0; v < L.nvar; ++v) U[v * L.sv + o] = b[v];
    } else {
      for (int v = 0; v < L.nvar; ++v) U[v * L.sv + o] = a[v];
    }
  }
}

template <int ND>
__global__ void unpack_kernel(Layout L, Phys P, const double* __restrict__ U, double* __restrict__ dst, int to_prim) {
  const long long ncell = (long long)L.n[0] * L.n[1] * L.n[2];
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < ncell; t += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(t % L.n[0]);
    const int j = (int)((t / L.n[0]) % L.n[1]);
    const int k = (int)(t / ((long long)L.n[0] * L.n[1]));
    const long long o = L.off(i + L.ng[0], j + L.ng[1], k + L.ng[2]);
    double a[NVMAX], b[NVMAX];
    for (int v = 0; v < L.nvar; ++v) a[v] = U[v * L.sv + o];
    if (to_prim) {
      cons_to_prim<ND>(P, L.nvar, a, b);
      for (int v = 0; v < L.nvar; ++v) dst[v * ncell + t] = b[v];
    } else {
      for (int v = 0; v < L.nvar; ++v) dst[v * ncell + t] = a[v];
    }
  }
}

static unsigned grid_for(long long work, int block) {
  long long g = (work + block - 1) / block;
  if (g > 148LL * 32) g = 148LL * 32;
  if (g < 1) g = 1;
  return (unsigned)g;
}

cudaError_t launch_pack(const Layout& L, const Phys& P, const double* src, double* U, int to_cons, cudaStream_t s) {
  const long long ncell = (long long)L.n[0] * L.n[1] * L.n[2];
  const unsigned g = grid_for(ncell, 256);
  if (L.ndim == 1) pack_kernel<1><<<g, 256, 0, s>>>(L, P, src, U, to_cons);
  else if (L.ndim == 2) pack_kernel<2><<<g, 256, 0, s>>>(L, P, src, U, to_cons);
  else pack_kernel<3><<<g, 256, 0, s>>>(L, P, src, U, to_cons);
  return cudaGetLastError();
}

cudaError_t launch_unpack(const Layout& L, const Phys& P, const double* U, double* dst, int to_prim, cudaStream_t s) {
  const long long ncell = (long long)L.n[0] * L.n[1] * L.n[2];
  const unsigned g = grid_for(ncell, 256);
  if (L.ndim == 1) unpack_kernel<1><<<g, 256, 0, s>>>(L, P, U, dst, to_prim);
  else if (L.ndim == 2) unpack_kernel<2><<<g, 256, 0, s>>>(L, P, U, dst, to_prim);
  else unpack_kernel<3><<<g, 256, 0, s>>>(L, P, U, dst, to_prim);
  return cudaGetLastError();
}

// A7 stand-alone: max over interior cells of sum_d (|u_d| + c_s)/l_d, warp shuffles + one
// block-level pass + one atomicMax per block.  Also flags rho <= 0, P <= 0, non-finite.
template <int ND>
__global__ void rate_kernel(Layout L, Tables T, Phys P, const double* __restrict__ U, unsigned long long* rate_bits, int* status) {
  const long long ncell = (long long)L.n[0] * L.n[1] * L.n[2];
  double rmax = 0.0;
  bool bad = false;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < ncell; t += (long long)gridDim.x * blockDim.x) {
    const int pi = (int)(t % L.n[0]) + L.ng[0];
    const int pj = (int)((t / L.n[0]) % L.n[1]) + L.ng[1];
    const int pk = (int)(t / ((long long)L.n[0] * L.n[1])) + L.ng[2];
    const long long o = L.off(pi, pj, pk);
    const double rho = U[o];
    const double ir = 1.0 / rho;
    double u[ND], u2 = 0.0;
#pragma unroll
    for (int d = 0; d < ND; ++d) {
      u[d] = U[(1 + d) * L.sv + o] * ir;
      u2 += u[d] * u[d];
    }
    const double p = P.gm1 * (U[(1 + ND) * L.sv + o] - 0.5 * rho * u2);
    if (!(rho > 0.0) || !(p > 0.0) || !isfinite(rho) || !isfinite(p)) {
      bad = true;
      continue;
    }
    const double cs = sqrt(P.gamma * p * ir);
    double rate = 0.0;
#pragma unroll
    for (int d = 0; d < ND; ++d) rate += (fabs(u[d]) + cs) * (T.lf[d][0][pi] * T.lf[d][1][pj] * T.lf[d][2][pk]);
    if (!isfinite(rate)) bad = true;
    else rmax = fmax(rmax, rate);
  }
  if (bad) atomicOr(status, 1);
  block_rate_max(rmax, rate_bits);
}

cudaError_t launch_rate(const Layout& L, const Tables& T, const Phys& P, const double* U, unsigned long long* rate_bits, int* status,
                        cudaStream_t s) {
  const long long ncell = (long long)L.n[0] * L.n[1] * L.n[2];
  long long g = (ncell + 255) / 256;
  if (g > 148LL * 8) g = 148LL * 8;
  if (L.ndim == 1) rate_kernel<1><<<(unsigned)g, 256, 0, s>>>(L, T, P, U, rate_bits, status);
  else if (L.ndim == 2) rate_kernel<2><<<(unsigned)g, 256, 0, s>>>(L, T, P, U, rate_bits, status);
  else rate_kernel<3><<<(unsigned)g, 256, 0, s>>>(L, T, P, U, rate_bits, status);
  return cudaGetLastError();
}

}  // namespace hx

// hx_aux.cu -- ghost / boundary fill (A0), pack / unpack between the caller's interior buffer and
// the padded arrays (with optional prim <-> cons through the EOS), stand-alone CFL reduction (A7).
// PAPER.md L203 (boundary conditions), Eq. 5 (EOS), R2 (CFL), R16-R17 (ghost layers).
#include "hx_common.cuh"

namespace hx {

// Ghost fill (A0), all directions in ONE launch.  The ordered fill "direction 0, then 1, then 2, each pass
// spanning the ghosts of the earlier ones" gives every ghost cell the value of the interior
// cell found by mapping each out-of-range index back into the interior with that direction's boundary
// condition (periodic: wrap; null gradient: clamp; reflective: mirror and flip the normal momentum) -- the maps
// of different directions commute, so the composition is evaluated directly: one read, one write per ghost cell.
struct GhostBC {
  int lo[3], hi[3];
};

__device__ __forceinline__ int ghost_src(int i, int n, int bc_lo, int bc_hi, bool& flip) {
  if (i < 0) {
    const int g = -i;
    if (bc_lo == HX_BC_PERIODIC) return n - g;
    if (bc_lo == HX_BC_TRANSMISSIVE) return 0;
    flip = !flip;
    return g - 1;
  }
  if (i >= n) {
    const int g = i - n + 1;
    if (bc_hi == HX_BC_PERIODIC) return g - 1;
    if (bc_hi == HX_BC_TRANSMISSIVE) return n - 1;
    flip = !flip;
    return n - g;
  }
  return i;
}

// Work is organised by ROWS of the padded array (fixed field, q1, q2; x varies), so that the index arithmetic is per row:
//   * rows interior in directions 1 and 2 hold only their 2 ng0 x-ghost cells: ONE THREAD per row fills them (blocks [0, nb_int)).
//     These columns are the expensive part (one 64-byte DRAM burst and a read-for-ownership per 16 useful bytes: ncu, 512^3 x 7
//     fields: 0.92 GB of traffic for 0.36 GB of ghost data, 0.28 ms); the 3-D tile kernel therefore writes them itself from the
//     registers of its boundary threads, and the fill that follows it is launched with skip_x (nb_int = 0);
//   * rows that are ghost rows in direction 1 or 2 are ghost from end to end: ONE BLOCK per row copies it from its source row,
//     coalesced, the x-ghost cells inside taking the composed map.
// blockIdx.y = field.
__global__ void __launch_bounds__(256) ghost_fill_kernel(Layout L, double* __restrict__ U, GhostBC bc, int nb_int) {
  const int v = blockIdx.y;
  double* __restrict__ Uv = U + (long long)v * L.sv;
  const int n0 = L.n[0], n1 = L.n[1], n2 = L.n[2], g0 = L.ng[0], g1 = L.ng[1], g2 = L.ng[2];
  if ((int)blockIdx.x < nb_int) {
    // ---- rows interior in 1 and 2: the x-ghost cells ----
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n1 * n2 || g0 == 0) return;
    const int j = r % n1, k = r / n1;
    double* row = Uv + L.off(0, j + g1, k + g2);           // padded x index 0 of this row
    double val[2 * NG];
    bool neg[2 * NG];
#pragma unroll
    for (int c = 0; c < 2 * NG; ++c) {                      // ghosts below: padded 0..ng-1, above: n+ng..n+2ng-1
      const int q = c < NG ? c : n0 + c;
      bool flip = false;
      const int src = ghost_src(q - g0, n0, bc.lo[0], bc.hi[0], flip) + g0;
      neg[c] = flip && v == 1;
      val[c] = row[src];
    }
#pragma unroll
    for (int c = 0; c < 2 * NG; ++c) {
      const int q = c < NG ? c : n0 + c;
      row[q] = neg[c] ? -val[c] : val[c];
    }
    return;
  }
  // ---- ghost rows: enumerate (q1, q2) with q2 in its ghost range (all q1), then q2 interior with q1 in its ghost range ----
  int gr = blockIdx.x - nb_int;
  const int np1 = L.np[1];
  int q1, q2;
  const int rows_z = 2 * g2 * np1;                          // rows with a ghost q2
  if (gr < rows_z) {
    const int c = gr / np1;
    q1 = gr - c * np1;
    q2 = c < g2 ? c : n2 + c;
  } else {
    gr -= rows_z;
    const int c = gr % (2 * g1);
    q2 = gr / (2 * g1) + g2;
    q1 = c < g1 ? c : n1 + c;
  }
  bool f1 = false, f2 = false;
  const int s1 = ghost_src(q1 - g1, n1, bc.lo[1], bc.hi[1], f1) + g1;
  const int s2 = ghost_src(q2 - g2, n2, bc.lo[2], bc.hi[2], f2) + g2;
  const bool neg_row = (f1 && v == 2 && L.ndim >= 2) != (f2 && v == 3 && L.ndim >= 3);
  const double* __restrict__ src = Uv + L.off(0, s1, s2);
  double* __restrict__ dst = Uv + L.off(0, q1, q2);
  for (int q0 = threadIdx.x; q0 < L.np[0]; q0 += blockDim.x) {
    bool f0 = false;
    const int s0 = ghost_src(q0 - g0, n0, bc.lo[0], bc.hi[0], f0) + g0;
    const double val = src[s0];
    dst[q0] = (neg_row != (f0 && v == 1)) ? -val : val;
  }
}

// skip_x: the x-ghost cells of the rows interior in directions 1 and 2 are already filled (by the 3-D tile kernel)
cudaError_t launch_ghost_fill(const Layout& L, double* U, const int* bc_lo, const int* bc_hi, int skip_x, cudaStream_t s) {
  GhostBC bc;
  for (int d = 0; d < 3; ++d) {
    bc.lo[d] = bc_lo[d];
    bc.hi[d] = bc_hi[d];
  }
  const long long rows_int = (long long)L.n[1] * L.n[2];
  const long long rows_ghost = (long long)L.np[1] * L.np[2] - rows_int;
  const long long nb_int = (L.ng[0] > 0 && !skip_x) ? (rows_int + 255) / 256 : 0;
  const long long blocks = nb_int + rows_ghost;
  if (blocks == 0) return cudaSuccess;
  if (blocks >= (1LL << 31)) return cudaErrorInvalidValue;
  ghost_fill_kernel<<<dim3((unsigned)blocks, (unsigned)L.nvar), 256, 0, s>>>(L, U, bc, (int)nb_int);
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// Self-gravity (Eq. 4; R28): g_r(r_c,i) = -[G M_c + G (4 pi / dOmega) (sum_{i'<i} m_i'
// + m_i (r_c^3 - r_-^3)/(r_+^3 - r_-^3))] / r_c^2 with the shell masses m_i = sum_{j,k} rho dV of the CURRENT state.
// Stage 1: each block sums rho x (theta weight) x (phi weight) over a fixed set of (j,k) rows for 256 radial
// cells (coalesced along r); stage 2: one block adds the partial sums in block order (deterministic), scans
// over r and rewrites the radial acceleration table, ghost entries included (mirror image behind a reflecting
// face, R25; central mass only inside r_min; everything outside r_max).
// ---------------------------------------------------------------------------------------------
struct SelfGrav {
  const double* xf[3];   // padded face coordinates of the three axes (device)
  double* partial;       // [nrows_groups][n0]
  const double* weights; // theta weights cos(th-) - cos(th+) [n1], then phi widths [n2] (constant in time: computed once)
  double* grav_r;        // the table T.grav[0], np[0] entries
  double GM, G;
  int groups, bc_lo, bc_hi;
};

__global__ void shell_weights_kernel(Layout L, SelfGrav sg, double* w) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < L.n[1]) w[t] = cos(sg.xf[1][t + L.ng[1]]) - cos(sg.xf[1][t + L.ng[1] + 1]);
  else if (t < L.n[1] + L.n[2]) {
    const int k = t - L.n[1];
    w[t] = sg.xf[2][k + L.ng[2] + 1] - sg.xf[2][k + L.ng[2]];
  }
}

__global__ void shell_mass_partial_kernel(Layout L, const double* __restrict__ U, SelfGrav sg) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= L.n[0]) return;
  const int rows = L.n[1] * L.n[2];
  double acc = 0.0;
  for (int r = blockIdx.y; r < rows; r += gridDim.y) {
    const int j = r % L.n[1], k = r / L.n[1];
    const double wt = sg.weights[j], wp = sg.weights[L.n[1] + k];
    acc = fma(U[L.off(i + L.ng[0], j + L.ng[1], k + L.ng[2])], wt * wp, acc);
  }
  sg.partial[(size_t)blockIdx.y * L.n[0] + i] = acc;
}

__global__ void self_gravity_table_kernel(Layout L, SelfGrav sg) {
  extern __shared__ double sm[];            // m[n0], then g[n0]
  double* m = sm;
  double* g = sm + L.n[0];
  const int n0 = L.n[0];
  for (int i = threadIdx.x; i < n0; i += blockDim.x) {
    double s = 0.0;
    for (int b = 0; b < sg.groups; ++b) s += sg.partial[(size_t)b * n0 + i];
    const double rm = sg.xf[0][i + L.ng[0]], rp = sg.xf[0][i + L.ng[0] + 1];
    m[i] = s * ((rp * rp * rp - rm * rm * rm) / 3.0);
  }
  __syncthreads();
  __shared__ double mtot;
  if (threadIdx.x == 0) {
    const double PI = 3.14159265358979323846;
    const double domega = (cos(sg.xf[1][L.ng[1]]) - cos(sg.xf[1][L.ng[1] + L.n[1]])) * (sg.xf[2][L.ng[2] + L.n[2]] - sg.xf[2][L.ng[2]]);
    const double scale = sg.G * 4.0 * PI / domega;
    double below = 0.0;
    for (int i = 0; i < n0; ++i) {
      const double rm = sg.xf[0][i + L.ng[0]], rp = sg.xf[0][i + L.ng[0] + 1], rc = 0.5 * (rm + rp);
      const double frac = (rc * rc * rc - rm * rm * rm) / (rp * rp * rp - rm * rm * rm);
      g[i] = -(sg.GM + scale * (below + m[i] * frac)) / (rc * rc);
      below += m[i];
    }
    mtot = sg.GM + scale * below;
  }
  __syncthreads();
  for (int p = threadIdx.x; p < L.np[0]; p += blockDim.x) {
    const int i = p - L.ng[0];
    const double rc = 0.5 * (sg.xf[0][p] + sg.xf[0][p + 1]);
    const bool refl_lo = sg.bc_lo == HX_BC_REFLECTING || sg.bc_lo == HX_BC_WEDGE, refl_hi = sg.bc_hi == HX_BC_REFLECTING || sg.bc_hi == HX_BC_WEDGE;
    double v;
    if (i < 0) v = refl_lo ? -g[-1 - i] : -sg.GM / (rc * rc);
    else if (i >= n0) v = refl_hi ? -g[2 * n0 - 1 - i] : -mtot / (rc * rc);
    else v = g[i];
    sg.grav_r[p] = v;
  }
}

// weights: n1 + n2 doubles of device memory; *weights_ready: filled on the first call (the angular weights do not change in time)
cudaError_t launch_self_gravity(const Layout& L, const double* U, const double* const xf[3], double* partial, int groups, double* grav_r,
                                double GM, double G, int bc_lo, int bc_hi, double* weights, bool* weights_ready, cudaStream_t s) {
  SelfGrav sg;
  for (int d = 0; d < 3; ++d) sg.xf[d] = xf[d];
  sg.partial = partial;
  sg.weights = weights;
  if (!*weights_ready) {
    const int nw = L.n[1] + L.n[2];
    shell_weights_kernel<<<(nw + 255) / 256, 256, 0, s>>>(L, sg, weights);
    if (cudaGetLastError() != cudaSuccess) return cudaErrorLaunchFailure;
    *weights_ready = true;
  }
  sg.grav_r = grav_r;
  sg.GM = GM;
  sg.G = G;
  sg.groups = groups;
  sg.bc_lo = bc_lo;
  sg.bc_hi = bc_hi;
  dim3 grid((unsigned)((L.n[0] + 255) / 256), (unsigned)groups);
  shell_mass_partial_kernel<<<grid, 256, 0, s>>>(L, U, sg);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const size_t smem = 2 * (size_t)L.n[0] * sizeof(double);
  if (smem > 48 * 1024) {
    e = cudaFuncSetAttribute(self_gravity_table_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  self_gravity_table_kernel<<<1, 256, smem, s>>>(L, sg);
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
    const double p = eos_pressure(P, rho, U[(1 + ND) * L.sv + o] - 0.5 * rho * u2);
    if (!(rho > 0.0) || !(p > 0.0) || !isfinite(rho) || !isfinite(p)) {
      bad = true;
      continue;
    }
    const double cs = eos_sound_speed(P, rho, p);
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

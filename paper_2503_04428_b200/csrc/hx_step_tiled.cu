// hx_step_tiled.cu -- the fused 3-D step kernel (A1-A7 of SURVEY 8(a) in ONE pass over HBM).
//
// Design (B200, sm_100a):
//   * A CTA owns an (x,y) tile of up to 30 x TY cells and marches along z over a chunk of planes.
//     Warp r <-> row j0-1+r (rows -1 and TY are the predictor ring), lane l <-> cell i0-1+l
//     (lanes 0 and wx+1 are the ring), so every x-neighbour exchange (slopes, face states, fluxes)
//     is a warp shuffle; y-neighbours go through shared memory; z-neighbours stay in registers of
//     the marching thread.  Every predictor, every face flux is computed once per tile.
//   * Each plane (tile + 2 ghost layers, all fields) is staged by ONE TMA bulk-tensor copy
//     (cp.async.bulk.tensor.4d, SASS UTMALDG) into a 2-deep shared-memory ring and signalled with an
//     mbarrier; cons->prim runs in place, the plane is then the neighbour source for the next step.
//   * The predicted face states carry (rho, u, P, E, c_s); HLL/HLLC flux once per face; the update
//     of cell k is finished when the flux through its upper z face arrives one plane later and is
//     written once, coalesced.  Spherical / gravity sources and the CFL rate of the new state are
//     folded in; the CTA reduces the rate with warp shuffles and issues one atomicMax.
//   * fp64 throughout; reciprocal and square root are MUFU seeds + Newton steps (<= 2 ulp, no slow
//     paths) because the FP64 pipe is the binding unit (DESIGN.md roofline).
//
// PAPER.md: Eq. 17 (slopes), Eq. 18 + Toro 16.5 (unsplit predictor), Eq. 19 (update), L201 (HLL/HLLC),
// Eq. 13-16 (spherical sources), Eq. 2-3 (gravity); readings R1-R25.
#include <cuda.h>

#include "hx_common.cuh"

namespace hx {

constexpr int BX = 34;   // tile box width: 30 cells + ring + one more ghost on each side (34*8 B = 17*16 B)
constexpr int TXMAX = 30;

struct TiledArgs {
  StepArgs s;
  int wx, wy;        // owner cells per tile in x (<= 30) and y (<= TY)
  int zc;            // planes per z chunk
};

// ------------------------------------------------------------------------------------------------
// fp64 helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double rcp_fast(double x) {   // 1/x, MUFU.RCP64H seed + 2 Newton steps
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y, 1.0);
  y = fma(y, e, y);
  e = fma(-x, y, 1.0);
  return fma(y, e, y);
}

__device__ __forceinline__ double sqrt_fast(double x) {  // sqrt(x), x > 0: MUFU.RSQ64H seed + coupled Newton
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double g = x * y, h = 0.5 * y;
  double r = fma(-h, g, 0.5);
  g = fma(g, r, g);
  h = fma(h, r, h);
  r = fma(-h, g, 0.5);
  g = fma(g, r, g);
  r = fma(-g, g, x);          // final correction: g += (x - g^2) * h
  return fma(r, h, g);
}

template <int LIM>
__device__ __forceinline__ double slope(int lim_rt, double a, double b) {
  if (LIM == HX_LIM_NONE) return 0.0;
  if (LIM == HX_LIM_MINMOD) {
    const double m = fmin(fabs(a), fabs(b));
    return (a * b > 0.0) ? copysign(m, a) : 0.0;
  }
  if (LIM == HX_LIM_MC) {
    const double fa = fabs(a), fb = fabs(b);
    const double m = fmin(fmin(fa + fa, fb + fb), 0.5 * (fa + fb));
    return (a * b > 0.0) ? copysign(m, a) : 0.0;
  }
  return limited_slope(lim_rt, a, b);
}

// ------------------------------------------------------------------------------------------------
// TMA / mbarrier PTX
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra.uni WAIT_DONE;\n"
      "bra.uni WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_plane(const CUtensorMap* tmap, void* dst, uint64_t* bar, int x, int y, int z) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(
          smem_u32(dst)),
      "l"(tmap), "r"(x), "r"(y), "r"(z), "r"(0), "r"(smem_u32(bar))
      : "memory");
}

// Face-state record exchanged between cells: predicted primitives + total energy + sound speed.
// index: 0 rho, 1..3 u, 4 P, 5 E, 6 c, 7.. scalars
template <int NV>
struct FS {
  static constexpr int N = NV + 2;
  double q[N];
};

// Predicted state on one face: primitives Wf = W + sgn*hw*sig (Eq. 17), conserved + dU (Eq. 18),
// back to primitives, plus E and c for the Riemann solver.  Also returns the analytic flux of the
// UNpredicted face state along dir (for the predictor sum) when WANT_FLUX.
template <int NV>
__device__ __forceinline__ void face_prims(const double* W, const double* sig, double shw, double* Wf) {
#pragma unroll
  for (int v = 0; v < NV; ++v) Wf[v] = fma(shw, sig[v], W[v]);
}

// conserved face state (rho, m[3], E, rho f) and its analytic flux along dir
template <int NV>
__device__ __forceinline__ void cons_and_flux(const Phys& P, int dir, const double* Wf, double* Uf, double* Ff) {
  const double r = Wf[0];
  Uf[0] = r;
  Uf[1] = r * Wf[1];
  Uf[2] = r * Wf[2];
  Uf[3] = r * Wf[3];
  const double ke = 0.5 * (Uf[1] * Wf[1] + Uf[2] * Wf[2] + Uf[3] * Wf[3]);
  Uf[4] = fma(Wf[4], P.igm1, ke);
  const double un = Wf[1 + dir];
  Ff[0] = Uf[1 + dir];
  Ff[1] = Uf[1] * un;
  Ff[2] = Uf[2] * un;
  Ff[3] = Uf[3] * un;
  Ff[1 + dir] += Wf[4];
  Ff[4] = (Uf[4] + Wf[4]) * un;
#pragma unroll
  for (int s = 5; s < NV; ++s) {
    Uf[s] = r * Wf[s];
    Ff[s] = Uf[s] * un;
  }
}

template <int NV>
__device__ __forceinline__ void predicted_state(const Phys& P, const double* Uf, const double* dU, FS<NV>& o) {
  const double r = Uf[0] + dU[0];
  const double ir = rcp_fast(r);
  const double m1 = Uf[1] + dU[1], m2 = Uf[2] + dU[2], m3 = Uf[3] + dU[3];
  const double E = Uf[4] + dU[4];
  const double u1 = m1 * ir, u2 = m2 * ir, u3 = m3 * ir;
  const double p = P.gm1 * (E - 0.5 * (m1 * u1 + m2 * u2 + m3 * u3));
  o.q[0] = r;
  o.q[1] = u1;
  o.q[2] = u2;
  o.q[3] = u3;
  o.q[4] = p;
  o.q[5] = E;
  o.q[6] = sqrt_fast(P.gamma * p * ir);
#pragma unroll
  for (int s = 5; s < NV; ++s) o.q[2 + s] = (Uf[s] + dU[s]) * ir;
}

// HLL / HLLC flux along dir from two face-state records (L | R).  F: rho, m[3], E, scalars.
template <int NV, int RS>
__device__ __forceinline__ void riemann_fs(const Phys& P, int dir, const FS<NV>& L, const FS<NV>& R, double* F) {
  const double uL = L.q[1 + dir], uR = R.q[1 + dir];
  const double SL = fmin(uL - L.q[6], uR - R.q[6]);
  const double SR = fmax(uL + L.q[6], uR + R.q[6]);
  const bool hllc = (RS == HX_RIEMANN_HLLC) || (RS < 0 && P.riemann == HX_RIEMANN_HLLC);
  if (hllc) {
    const double mL = L.q[0] * (SL - uL), mR = R.q[0] * (SR - uR);
    const double Ss = (R.q[4] - L.q[4] + uL * mL - uR * mR) * rcp_fast(mL - mR);
    const bool left = (SL >= 0.0) || (Ss >= 0.0);
    const bool upwind = (SL >= 0.0) || (!left && SR <= 0.0);   // pure F_L or F_R
    const double SK = left ? SL : SR, mK = left ? mL : mR, uK = left ? uL : uR;
    double qk[FS<NV>::N];
#pragma unroll
    for (int v = 0; v < FS<NV>::N; ++v) qk[v] = left ? L.q[v] : R.q[v];
    const double rK = qk[0], pK = qk[4], EK = qk[5];
    const double w = rcp_fast(SK - Ss);
    const double fac = mK * w;                      // rho*_K
    const double fr = rK * uK;                      // mass flux of side K
    const double SKe = upwind ? 0.0 : SK;
    const double dr = fac - rK;
    F[0] = fma(SKe, dr, fr);
    double Fm[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) Fm[d] = fma(SKe, dr * qk[1 + d], fr * qk[1 + d]);
    // normal component: F_K + S_K (rho* S* - rho_K u_K)
    Fm[dir] = fma(SKe, fma(fac, Ss, -fr), fma(fr, uK, pK));
    F[1] = Fm[0];
    F[2] = Fm[1];
    F[3] = Fm[2];
    const double Es = fma((SK - uK) * w, EK, (Ss - uK) * fma(fac, Ss, pK * w));   // E*_K
    F[4] = fma(SKe, Es - EK, (EK + pK) * uK);
#pragma unroll
    for (int s = 5; s < NV; ++s) F[s] = F[0] * qk[2 + s];   // passive scalars ride the mass flux (R7)
  } else {
    // HLL: (SR F_L - SL F_R + SL SR (U_R - U_L)) / (SR - SL), upwind flux outside the fan
    const bool useL = SL >= 0.0, useR = (!useL) && SR <= 0.0;
    const double iw = rcp_fast(SR - SL);
    const double aL = useL ? 1.0 : (useR ? 0.0 : SR * iw), aR = useL ? 0.0 : (useR ? 1.0 : -SL * iw);
    const double dd = (useL || useR) ? 0.0 : SL * SR * iw;
    const double frL = L.q[0] * uL, frR = R.q[0] * uR;
    F[0] = aL * frL + aR * frR + dd * (R.q[0] - L.q[0]);
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const double mL = L.q[0] * L.q[1 + d], mR = R.q[0] * R.q[1 + d];
      const double fL = mL * uL + (d == dir ? L.q[4] : 0.0), fR = mR * uR + (d == dir ? R.q[4] : 0.0);
      F[1 + d] = aL * fL + aR * fR + dd * (mR - mL);
    }
    F[4] = aL * ((L.q[5] + L.q[4]) * uL) + aR * ((R.q[5] + R.q[4]) * uR) + dd * (R.q[5] - L.q[5]);
#pragma unroll
    for (int s = 5; s < NV; ++s) {
      const double sL = L.q[0] * L.q[2 + s], sR = R.q[0] * R.q[2 + s];
      F[s] = aL * (sL * uL) + aR * (sR * uR) + dd * (sR - sL);
    }
  }
}

template <int NV>
__device__ __forceinline__ void prim_of_cons(const Phys& P, const double* U, double* W) {
  const double ir = rcp_fast(U[0]);
  W[0] = U[0];
  W[1] = U[1] * ir;
  W[2] = U[2] * ir;
  W[3] = U[3] * ir;
  W[4] = P.gm1 * (U[4] - 0.5 * (U[1] * W[1] + U[2] * W[2] + U[3] * W[3]));
#pragma unroll
  for (int s = 5; s < NV; ++s) W[s] = U[s] * ir;
}

template <int N>
__device__ __forceinline__ void shfl_up_vec(const double* in, double* out) {
#pragma unroll
  for (int v = 0; v < N; ++v) out[v] = __shfl_up_sync(0xffffffffu, in[v], 1);
}
template <int N>
__device__ __forceinline__ void shfl_down_vec(const double* in, double* out) {
#pragma unroll
  for (int v = 0; v < N; ++v) out[v] = __shfl_down_sync(0xffffffffu, in[v], 1);
}

// ------------------------------------------------------------------------------------------------
// The kernel
// ------------------------------------------------------------------------------------------------
template <int NV, int TY>
struct TileSmem {
  static constexpr int BY = TY + 4;
  static constexpr int ROWS = TY + 2;
  static constexpr int NF = NV + 2;
  static constexpr size_t plane_bytes = (size_t)NV * BY * BX * sizeof(double);
  static constexpr size_t plane_stride = (plane_bytes + 127) / 128 * 128;
  static constexpr size_t yp_bytes = (size_t)NF * ROWS * 32 * sizeof(double);
  static constexpr size_t fy_bytes = (size_t)NV * ROWS * 32 * sizeof(double);
  static constexpr size_t total = 2 * plane_stride + yp_bytes + fy_bytes + 64 + 128;
};

template <int NV, bool SPH, bool GRAV, int LIM, int RS, int TY>
__global__ void __launch_bounds__((TY + 2) * 32, 1)
step_tiled3d_kernel(const __grid_constant__ CUtensorMap tmap, const TiledArgs a) {
  using SM = TileSmem<NV, TY>;
  constexpr int BY = SM::BY, ROWS = SM::ROWS, NF = SM::NF;
  extern __shared__ unsigned char smem_raw[];
  unsigned char* base = (unsigned char*)(((uintptr_t)smem_raw + 127) & ~(uintptr_t)127);
  double* plane[2] = {(double*)base, (double*)(base + SM::plane_stride)};
  double* ypbuf = (double*)(base + 2 * SM::plane_stride);
  double* fybuf = (double*)(base + 2 * SM::plane_stride + SM::yp_bytes);
  uint64_t* mbar = (uint64_t*)(base + 2 * SM::plane_stride + SM::yp_bytes + SM::fy_bytes);

  const StepArgs& s = a.s;
  const Layout& L = s.L;
  const Tables& T = s.T;
  const Phys& P = s.P;
  const int lane = threadIdx.x & 31, row = threadIdx.x >> 5;
  const int i0 = blockIdx.x * a.wx, j0 = blockIdx.y * a.wy;
  const int k0 = blockIdx.z * a.zc, k1 = min(L.n[2], k0 + a.zc);
  const int i = i0 + lane - 1, j = j0 + row - 1;           // interior indices of this thread's column
  // padded indices for the 1-D tables, clamped so that idle lanes read valid table entries
  const int pi = min(max(i + NG, 1), L.np[0] - 2), pj = min(max(j + NG, 1), L.np[1] - 2);
  const bool owner = lane >= 1 && lane <= a.wx && i < L.n[0] && row >= 1 && row <= a.wy && j < L.n[1];
  const int bx = lane + 1, by = row + 1;                    // position inside the tile box
  const int cidx = by * BX + bx;                            // offset inside one field of a plane
  constexpr int FSTR = BY * BX;                             // field stride inside a plane
  const int eidx = row * 32 + lane;                         // offset inside one field of ypbuf / fybuf

  // loop-invariant geometry of this column (products of 1-D tables)
  const double idx_lo = T.idx[0][pi], idx_hi = T.idx[0][pi + 1], hwx = T.hw[0][pi];
  const double idy_lo = T.idx[1][pj], idy_hi = T.idx[1][pj + 1], hwy = T.hw[1][pj];
  const double cm0 = T.cf[0][0][0][pi] * T.cf[0][0][1][pj], cp0 = T.cf[0][1][0][pi] * T.cf[0][1][1][pj];
  const double cm1 = T.cf[1][0][0][pi] * T.cf[1][0][1][pj], cp1 = T.cf[1][1][0][pi] * T.cf[1][1][1][pj];
  const double c2m = T.cf[2][0][0][pi] * T.cf[2][0][1][pj], c2p = T.cf[2][1][0][pi] * T.cf[2][1][1][pj];
  const double il0 = T.lf[0][0][pi] * T.lf[0][1][pj], il1 = T.lf[1][0][pi] * T.lf[1][1][pj], il2ij = T.lf[2][0][pi] * T.lf[2][1][pj];
  const double gx = GRAV ? T.grav[0][pi] : 0.0, gy = GRAV ? T.grav[1][pj] : 0.0;
  const double dt = s.dt, hdt = 0.5 * s.dt;

  const int xs = i0 + L.lead, ys = j0;                     // box origin in storage coordinates (cell i0-2, j0-2)
  uint32_t phase[2] = {0u, 0u};
  if (threadIdx.x == 0) {
    mbar_init(&mbar[0], 1);
    mbar_init(&mbar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (threadIdx.x == 0) {   // planes k0-2 and k0-1 (padded z index = interior + NG)
    mbar_expect_tx(&mbar[0], (uint32_t)SM::plane_bytes);
    tma_load_plane(&tmap, plane[0], &mbar[0], xs, ys, k0 - 2 + NG);
    mbar_expect_tx(&mbar[1], (uint32_t)SM::plane_bytes);
    tma_load_plane(&tmap, plane[1], &mbar[1], xs, ys, k0 - 1 + NG);
  }

  // converts the cell at box offset `off` of plane `pl` in place (raw conserved -> primitive)
  auto convert_in_place = [&](double* pl, int off, double* Wout) {
    double U[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) U[v] = pl[v * FSTR + off];
    prim_of_cons<NV>(P, U, Wout);
#pragma unroll
    for (int v = 0; v < NV; ++v) pl[v * FSTR + off] = Wout[v];
  };
  // own cell + the second ghost layer cells this thread is responsible for
  auto convert_plane = [&](double* pl, double* Wown) {
    convert_in_place(pl, cidx, Wown);
    double tmp[NV];
    if (lane == 0) convert_in_place(pl, cidx - 1, tmp);
    if (lane == 31) convert_in_place(pl, cidx + 1, tmp);
    if (row == 0) convert_in_place(pl, cidx - BX, tmp);
    if (row == ROWS - 1) convert_in_place(pl, cidx + BX, tmp);
  };

  double Wc[NV], az[NV];      // W(p) of this column; backward z gradient (W(p) - W(p-1)) / dz
  {
    double Wm2[NV];
    mbar_wait(&mbar[0], phase[0]);
    phase[0] ^= 1u;
#pragma unroll
    for (int v = 0; v < NV; ++v) Wm2[v] = plane[0][v * FSTR + cidx];
    {
      double U[NV];
#pragma unroll
      for (int v = 0; v < NV; ++v) U[v] = Wm2[v];
      prim_of_cons<NV>(P, U, Wm2);
    }
    __syncthreads();          // everyone has read plane k0-2: its buffer can be refilled
    if (threadIdx.x == 0) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(&mbar[0], (uint32_t)SM::plane_bytes);
      tma_load_plane(&tmap, plane[0], &mbar[0], xs, ys, k0 + NG);
    }
    mbar_wait(&mbar[1], phase[1]);
    phase[1] ^= 1u;
    convert_plane(plane[1], Wc);
    const double idz = __ldg(T.idx[2] + (k0 - 1 + NG));
#pragma unroll
    for (int v = 0; v < NV; ++v) az[v] = (Wc[v] - Wm2[v]) * idz;
    __syncthreads();
  }

  FS<NV> zp;                  // predicted state on the upper z face of the previous plane
  double Up[NV];              // partially updated cell of the previous plane
  double Un0 = 0.0, Unm[3] = {0.0, 0.0, 0.0};   // rho^n, m^n of the previous plane (time-centred gravity)
  double rate_max = 0.0;
  bool bad = false;
#pragma unroll
  for (int v = 0; v < NF; ++v) zp.q[v] = 1.0;
#pragma unroll
  for (int v = 0; v < NV; ++v) Up[v] = 1.0;

  int cur = 1;                // plane[cur] holds W(p); plane[cur^1] receives raw(p+1)
  for (int p = k0 - 1; p <= k1; ++p) {
    const int pk = p + NG;
    const int nxt = cur ^ 1;
    const bool do_xy = (p >= k0) && (p < k1);
    double* Pc = plane[cur];
    double* Pn = plane[nxt];
    // ---- plane p+1 arrives: convert in place --------------------------------------------------
    double Wn[NV];
    mbar_wait(&mbar[nxt], phase[nxt]);
    phase[nxt] ^= 1u;
    convert_plane(Pn, Wn);

    // per-plane z geometry (uniform addresses: broadcast loads)
    const double idz_hi = __ldg(T.idx[2] + pk + 1), hwz = __ldg(T.hw[2] + pk);
    const double cm2 = c2m * __ldg(T.cf[2][0][2] + pk), cp2 = c2p * __ldg(T.cf[2][1][2] + pk);
    const double gz = GRAV ? __ldg(T.grav[2] + pk) : 0.0;

    // ---- O2 limited slopes ---------------------------------------------------------------------
    double sx[NV], sy[NV], sz[NV];
    {
      double Wxp[NV], bxg[NV], axg[NV];
      shfl_down_vec<NV>(Wc, Wxp);
      if (lane == 31) {
#pragma unroll
        for (int v = 0; v < NV; ++v) Wxp[v] = Pc[v * FSTR + cidx + 1];
      }
#pragma unroll
      for (int v = 0; v < NV; ++v) bxg[v] = (Wxp[v] - Wc[v]) * idx_hi;
      shfl_up_vec<NV>(bxg, axg);
      if (lane == 0) {
#pragma unroll
        for (int v = 0; v < NV; ++v) axg[v] = (Wc[v] - Pc[v * FSTR + cidx - 1]) * idx_lo;
      }
#pragma unroll
      for (int v = 0; v < NV; ++v) sx[v] = slope<LIM>(P.limiter, axg[v], bxg[v]);
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const double wm = Pc[v * FSTR + cidx - BX], wp = Pc[v * FSTR + cidx + BX];
        sy[v] = slope<LIM>(P.limiter, (Wc[v] - wm) * idy_lo, (wp - Wc[v]) * idy_hi);
      }
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const double b = (Wn[v] - Wc[v]) * idz_hi;
        sz[v] = slope<LIM>(P.limiter, az[v], b);
        az[v] = b;
      }
    }

    // ---- O3/O4: face states, half-step increment dU (Eq. 17-18, unsplit) -------------------------
    double Uxm[NV], Uxp[NV], Uym[NV], Uyp[NV], Uzm[NV], Uzp[NV], dU[NV];
    {
      double Wf[NV], Ff[NV];
      face_prims<NV>(Wc, sx, -hwx, Wf);
      cons_and_flux<NV>(P, 0, Wf, Uxm, Ff);
#pragma unroll
      for (int v = 0; v < NV; ++v) dU[v] = Ff[v] * cm0;
      face_prims<NV>(Wc, sx, hwx, Wf);
      cons_and_flux<NV>(P, 0, Wf, Uxp, Ff);
#pragma unroll
      for (int v = 0; v < NV; ++v) dU[v] = fma(-Ff[v], cp0, dU[v]);
      face_prims<NV>(Wc, sy, -hwy, Wf);
      cons_and_flux<NV>(P, 1, Wf, Uym, Ff);
#pragma unroll
      for (int v = 0; v < NV; ++v) dU[v] = fma(Ff[v], cm1, dU[v]);
      face_prims<NV>(Wc, sy, hwy, Wf);
      cons_and_flux<NV>(P, 1, Wf, Uyp, Ff);
#pragma unroll
      for (int v = 0; v < NV; ++v) dU[v] = fma(-Ff[v], cp1, dU[v]);
      face_prims<NV>(Wc, sz, -hwz, Wf);
      cons_and_flux<NV>(P, 2, Wf, Uzm, Ff);
#pragma unroll
      for (int v = 0; v < NV; ++v) dU[v] = fma(Ff[v], cm2, dU[v]);
      face_prims<NV>(Wc, sz, hwz, Wf);
      cons_and_flux<NV>(P, 2, Wf, Uzp, Ff);
#pragma unroll
      for (int v = 0; v < NV; ++v) dU[v] = fma(-Ff[v], cp2, dU[v]);
    }
    const double rho = Wc[0];
    const double mcx = rho * Wc[1], mcy = rho * Wc[2], mcz = rho * Wc[3];
    if (SPH) {   // cell-centred geometric sources (R8)
      const double ur = Wc[1], ut = Wc[2], up = Wc[3], pr = Wc[4];
      const double Ar = __ldg(T.Ar + pi), crg = __ldg(T.cr + pi);
      dU[1] += (mcy * ut + mcz * up + 2.0 * pr) * __ldg(T.gr + pi);
      dU[2] += -mcy * ur * Ar + (mcz * up + pr) * crg * __ldg(T.gt + pj);
      dU[3] += -mcz * ur * Ar - mcz * ut * crg * __ldg(T.At + pj);
    }
    if (GRAV) {
      dU[1] = fma(rho, gx, dU[1]);
      dU[2] = fma(rho, gy, dU[2]);
      dU[3] = fma(rho, gz, dU[3]);
      dU[4] += mcx * gx + mcy * gy + mcz * gz;
    }
    if (LIM == HX_LIM_NONE || (LIM < 0 && P.limiter == HX_LIM_NONE)) {   // R19: no predictor
#pragma unroll
      for (int v = 0; v < NV; ++v) dU[v] = 0.0;
    } else {
#pragma unroll
      for (int v = 0; v < NV; ++v) dU[v] *= hdt;
    }

    // conserved U^n of this cell (for the update) and P-bar of the centred predicted state
    double Un[NV];
    Un[0] = rho;
    Un[1] = mcx;
    Un[2] = mcy;
    Un[3] = mcz;
    Un[4] = fma(Wc[4], P.igm1, 0.5 * (mcx * Wc[1] + mcy * Wc[2] + mcz * Wc[3]));
#pragma unroll
    for (int v = 5; v < NV; ++v) Un[v] = rho * Wc[v];

    // ---- predicted face states ------------------------------------------------------------------
    FS<NV> fyp;
    predicted_state<NV>(P, Uyp, dU, fyp);
    if (do_xy) {
#pragma unroll
      for (int v = 0; v < NF; ++v) ypbuf[v * (ROWS * 32) + eidx] = fyp.q[v];
    }
    __syncthreads();                                   // (1) y+ states visible; all reads of plane[cur] done
    if (threadIdx.x == 0 && p + 2 <= k1 + 1) {         // refill plane[cur] with raw(p+2)
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(&mbar[cur], (uint32_t)SM::plane_bytes);
      tma_load_plane(&tmap, Pc, &mbar[cur], xs, ys, p + 2 + NG);
    }

    double acc[NV];                                    // sum of face-flux contributions of cell p (x, y, lower z)
#pragma unroll
    for (int v = 0; v < NV; ++v) acc[v] = 0.0;
    double Sr = 0.0, St = 0.0, Sp = 0.0;               // spherical source accumulators (Eq. 14-16)
    double rr_i = 0.0, st_j = 0.0, gr_i = 0.0, cgt = 0.0;
    if (SPH) {
      rr_i = __ldg(T.rr + pi);
      st_j = __ldg(T.st + pj);
      gr_i = __ldg(T.gr + pi);
      cgt = __ldg(T.cr + pi) * __ldg(T.gt + pj);
    }

    if (do_xy) {
      // ---- y faces: flux through j-1/2 here, through j+1/2 from the row above --------------------
      FS<NV> fl, fr;
      double F[NV], Fh[NV];
      predicted_state<NV>(P, Uym, dU, fr);
      const int em = (row > 0) ? eidx - 32 : eidx;
#pragma unroll
      for (int v = 0; v < NF; ++v) fl.q[v] = ypbuf[v * (ROWS * 32) + em];
      riemann_fs<NV, RS>(P, 1, fl, fr, F);
#pragma unroll
      for (int v = 0; v < NV; ++v) fybuf[v * (ROWS * 32) + eidx] = F[v];
#pragma unroll
      for (int v = 0; v < NV; ++v) acc[v] = F[v] * cm1;
      if (SPH) {
        Sr += 0.5 * F[2];
        Sp -= st_j * F[3] * cm1;
      }
      // ---- x faces via shuffles ---------------------------------------------------------------------
      {
        FS<NV> own;
        predicted_state<NV>(P, Uxp, dU, own);
        shfl_up_vec<NF>(own.q, fl.q);
        predicted_state<NV>(P, Uxm, dU, fr);
        riemann_fs<NV, RS>(P, 0, fl, fr, F);
        shfl_down_vec<NV>(F, Fh);
#pragma unroll
        for (int v = 0; v < NV; ++v) acc[v] += F[v] * cm0 - Fh[v] * cp0;
        if (SPH) {
          St -= rr_i * (Fh[2] * cp0 + F[2] * cm0);
          Sp -= rr_i * (Fh[3] * cp0 + F[3] * cm0);
        }
      }
      __syncthreads();                                 // (2) y fluxes visible
      const int ep = (row < ROWS - 1) ? eidx + 32 : eidx;
#pragma unroll
      for (int v = 0; v < NV; ++v) Fh[v] = fybuf[v * (ROWS * 32) + ep];
#pragma unroll
      for (int v = 0; v < NV; ++v) acc[v] = fma(-Fh[v], cp1, acc[v]);
      if (SPH) {
        Sr += 0.5 * Fh[2];
        Sp -= st_j * Fh[3] * cp1;
      }
    }

    // ---- z face p-1/2: previous plane's z+ state | this plane's z- state ---------------------------
    FS<NV> fzm;
    predicted_state<NV>(P, Uzm, dU, fzm);
    double Fz[NV];
    riemann_fs<NV, RS>(P, 2, zp, fzm, Fz);

    // ---- finish cell p-1 (its upper z flux is Fz) and write it once -----------------------------------
    if (p - 1 >= k0) {
      const double cpz_prev = c2p * __ldg(T.cf[2][1][2] + pk - 1);
      double Unew[NV];
#pragma unroll
      for (int v = 0; v < NV; ++v) Unew[v] = fma(-dt * cpz_prev, Fz[v], Up[v]);
      if (SPH) {   // phi-face part of the sources of cell p-1: 0.5 F^phi_phi on S_r and S_theta
        Unew[1] = fma(dt * gr_i, 0.5 * Fz[3], Unew[1]);
        Unew[2] = fma(dt * cgt, 0.5 * Fz[3], Unew[2]);
      }
      if (GRAV) {  // time-centred (R13)
        const double gzp = __ldg(T.grav[2] + pk - 1);
        const double hr = 0.5 * dt * (Un0 + Unew[0]);
        const double m1 = fma(hr, gx, Unew[1]), m2 = fma(hr, gy, Unew[2]), m3 = fma(hr, gzp, Unew[3]);
        Unew[4] += 0.5 * dt * ((Unm[0] + m1) * gx + (Unm[1] + m2) * gy + (Unm[2] + m3) * gzp);
        Unew[1] = m1;
        Unew[2] = m2;
        Unew[3] = m3;
      }
      if (owner) {
        const long long o = L.off(i + NG, j + NG, pk - 1);
#pragma unroll
        for (int v = 0; v < NV; ++v) s.Uout[v * L.sv + o] = Unew[v];
        // A7: CFL rate of the new state + positivity check
        const double ir = rcp_fast(Unew[0]);
        const double u1 = Unew[1] * ir, u2 = Unew[2] * ir, u3 = Unew[3] * ir;
        const double pn = P.gm1 * (Unew[4] - 0.5 * (Unew[1] * u1 + Unew[2] * u2 + Unew[3] * u3));
        if (!(Unew[0] > 0.0) || !(pn > 0.0) || !isfinite(Unew[0]) || !isfinite(pn)) {
          bad = true;
        } else {
          const double cs = sqrt_fast(P.gamma * pn * ir);
          const double il2 = il2ij * __ldg(T.lf[2][2] + pk - 1);
          const double rate = (fabs(u1) + cs) * il0 + (fabs(u2) + cs) * il1 + (fabs(u3) + cs) * il2;
          if (!isfinite(rate)) bad = true;
          else rate_max = fmax(rate_max, rate);
        }
      }
    }

    // ---- start cell p: U^n + dt * (x, y and lower z contributions) -------------------------------------
    if (do_xy) {
#pragma unroll
      for (int v = 0; v < NV; ++v) Up[v] = fma(dt, fma(Fz[v], cm2, acc[v]), Un[v]);
      if (SPH) {
        // theta / phi face parts known now; F^phi_phi lower-face half; P-bar is not needed in 3-D
        Up[1] = fma(dt, (Sr + 0.5 * Fz[3]) * gr_i, Up[1]);
        Up[2] = fma(dt, St + 0.5 * Fz[3] * cgt, Up[2]);
        Up[3] = fma(dt, Sp, Up[3]);
      }
      Un0 = Un[0];
      Unm[0] = Un[1];
      Unm[1] = Un[2];
      Unm[2] = Un[3];
    }
    predicted_state<NV>(P, Uzp, dU, zp);

    // ---- roll ---------------------------------------------------------------------------------------------
#pragma unroll
    for (int v = 0; v < NV; ++v) Wc[v] = Wn[v];
    cur = nxt;
  }

  if (bad) atomicOr(s.status, 1);
  block_rate_max(rate_max, s.rate_bits);
}

// ------------------------------------------------------------------------------------------------
// Host side: tensor maps, launch configuration
// ------------------------------------------------------------------------------------------------
struct TiledPlan {
  CUtensorMap tmap[2];
  int ty;
  int wx, wy, zc;
  dim3 grid;
  size_t smem;
  const char* name;
};

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

constexpr int TY_DEFAULT = 10;

static bool nv_supported(int nv) { return nv == 5 || nv == 6 || nv == 7 || nv == 9; }

int tiled_supported(const Layout& L, const Phys&) {
  return L.ndim == 3 && nv_supported(L.nvar) && L.n[0] >= 4 && L.n[1] >= 2 && L.n[2] >= 2;
}

template <int NV, bool SPH, bool GRAV, int LIM, int RS>
static cudaError_t launch_cfg(TiledPlan* plan, const TiledArgs& ta, int cur, cudaStream_t st) {
  auto kern = step_tiled3d_kernel<NV, SPH, GRAV, LIM, RS, TY_DEFAULT>;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TileSmem<NV, TY_DEFAULT>::total);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  kern<<<plan->grid, (TY_DEFAULT + 2) * 32, TileSmem<NV, TY_DEFAULT>::total, st>>>(plan->tmap[cur], ta);
  return cudaGetLastError();
}

template <int NV>
static cudaError_t launch_nv(TiledPlan* plan, const TiledArgs& ta, int cur, cudaStream_t st) {
  const Phys& P = ta.s.P;
  const bool sph = P.spherical != 0, grav = P.gravity != HX_GRAV_NONE;
  // the three measured configurations get fully specialised kernels; everything else the runtime-switch build
  if constexpr (NV == 5) {
    if (!sph && !grav && P.limiter == HX_LIM_MINMOD && P.riemann == HX_RIEMANN_HLLC)
      return launch_cfg<NV, false, false, HX_LIM_MINMOD, HX_RIEMANN_HLLC>(plan, ta, cur, st);
  }
  if constexpr (NV == 7) {
    if (!sph && grav && P.limiter == HX_LIM_MC && P.riemann == HX_RIEMANN_HLLC)
      return launch_cfg<NV, false, true, HX_LIM_MC, HX_RIEMANN_HLLC>(plan, ta, cur, st);
  }
  if constexpr (NV == 9) {
    if (sph && P.limiter == HX_LIM_MINMOD && P.riemann == HX_RIEMANN_HLLC)
      return launch_cfg<NV, true, true, HX_LIM_MINMOD, HX_RIEMANN_HLLC>(plan, ta, cur, st);
  }
  if (sph) return launch_cfg<NV, true, true, -1, -1>(plan, ta, cur, st);
  return launch_cfg<NV, false, true, -1, -1>(plan, ta, cur, st);
}

cudaError_t tiled_plan_create(const Layout& L, const Phys&, double* const U[2], TiledPlan** out) {
  *out = nullptr;
  EncodeTiledFn enc = get_encode_fn();
  if (!enc) return cudaErrorNotSupported;
  TiledPlan* p = new TiledPlan();
  p->ty = TY_DEFAULT;
  const int ntx = (L.n[0] + TXMAX - 1) / TXMAX, nty = (L.n[1] + p->ty - 1) / p->ty;
  p->wx = (L.n[0] + ntx - 1) / ntx;
  p->wx += p->wx & 1;   // even tile width: with the even `lead` every TMA box then starts on a 16-byte boundary
                        // (an odd start coordinate of this fp64 box raises "illegal instruction" on sm_100a)
  p->wy = (L.n[1] + nty - 1) / nty;
  // z chunks: enough CTAs for >= ~6 waves over 148 SMs, chunks of at least 16 planes (2 warm-up planes each)
  int nzc = 1;
  const long long cols = (long long)ntx * nty;
  while (cols * nzc < 148LL * 6 && L.n[2] / (nzc + 1) >= 16) ++nzc;
  p->zc = (L.n[2] + nzc - 1) / nzc;
  nzc = (L.n[2] + p->zc - 1) / p->zc;
  p->grid = dim3((unsigned)((L.n[0] + p->wx - 1) / p->wx), (unsigned)((L.n[1] + p->wy - 1) / p->wy), (unsigned)nzc);
  p->name = "tiled3d";
  for (int b = 0; b < 2; ++b) {
    const cuuint64_t dims[4] = {(cuuint64_t)L.sy, (cuuint64_t)L.np[1], (cuuint64_t)L.np[2], (cuuint64_t)L.nvar};
    const cuuint64_t strides[3] = {(cuuint64_t)L.sy * 8, (cuuint64_t)L.sz * 8, (cuuint64_t)L.sv * 8};
    const cuuint32_t box[4] = {(cuuint32_t)BX, (cuuint32_t)(p->ty + 4), 1u, (cuuint32_t)L.nvar};
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

void tiled_plan_destroy(TiledPlan* p) { delete p; }
const char* tiled_kernel_name(const TiledPlan* p) { return p ? p->name : "tiled3d"; }

cudaError_t launch_step_tiled(TiledPlan* plan, const StepArgs& a, int cur, cudaStream_t st) {
  TiledArgs ta;
  ta.s = a;
  ta.wx = plan->wx;
  ta.wy = plan->wy;
  ta.zc = plan->zc;
  switch (a.L.nvar) {
    case 5: return launch_nv<5>(plan, ta, cur, st);
    case 6: return launch_nv<6>(plan, ta, cur, st);
    case 7: return launch_nv<7>(plan, ta, cur, st);
    case 9: return launch_nv<9>(plan, ta, cur, st);
    default: return cudaErrorNotSupported;
  }
}

}  // namespace hx

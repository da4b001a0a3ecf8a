// hx_step_tile2d.cuh -- the fused 2-D step kernel (A1-A7 of SURVEY 8(a) in ONE pass), Cartesian grids.
//
// The 2-D counterpart of hx_step_tile2.cuh (config 2 of BASELINE.json, the Kelvin-Helmholtz run of PAPER.md
// Sect. 4.1; "1D, 2D, or 3D", L149).  Same design, one dimension down:
//   * a CTA owns a strip of NW x 32 = 352 cells in x (warp <-> 32-cell segment, lane <-> cell) and marches along y over a
//     chunk of rows; a row (strip + 2 ghost cells on each side, all fields) arrives by TWO TMA bulk-tensor copies (a box is at
//     most 256 elements wide) into a 3-deep ring signalled by mbarriers; cons -> prim runs in place;
//   * y is the march direction: the y slopes, the predicted y+ state of the previous row and the partially updated
//     cell of the previous row stay in registers;
//   * x neighbours exchange through shared memory: a cell writes the predicted state of its x+ face into its own
//     slot, the neighbour across that face solves the Riemann problem ONCE and writes the flux back into the same
//     slot; the slots are double buffered by row parity so that ONE CTA-wide barrier per row suffices;
//   * the two cells of the one-cell ring left and right of the strip are handled by two lanes of one extra warp; with eleven
//     owner warps it completes the third warpgroup, so that every scheduler holds three warps (a ring warp in a warpgroup of its
//     own, rebalanced with setmaxnreg as in 3-D, leaves one scheduler with one warp more than the others: measured slower);
//   * the CFL rate of a cell is folded in one row after it was written (A7), reduced by warp shuffles, one atomicMax
//     per CTA.
// Pointwise arithmetic as in the 3-D kernel (reciprocal / square root = MUFU seed + cubic correction, limiters on
// pre-scaled one-sided differences, flux differences accumulated into the half-step increment, tangential momentum
// and scalar fluxes as value x mass flux), written for two velocity components.
//
// PAPER.md: Eq. 17 (slopes), Eq. 18 + Toro 16.5 (unsplit predictor), Eq. 19 (update), L201 (HLL/HLLC), Eq. 2
// (uniform gravity), Eq. 5 (ideal gas); readings R1-R25.  Spherical 2-D grids, the gas + radiation EOS and
// the internal-energy monitoring run on the generic kernel.
#pragma once
#include "hx_step_tile2.cuh"

namespace hx {
namespace t2d {

using t2::dmax;
using t2::dmin;
using t2::lim_pre;
using t2::lim_pre_n;
using t2::lim_scale;
using t2::mbar_expect_tx;
using t2::mbar_init;
using t2::mbar_wait;
using t2::rcp3;
using t2::rcp3_n;
using t2::smem_u32;
using t2::sqrt3;
using t2::sqrt3_n;

#ifndef HX_T2D_NW
#define HX_T2D_NW 11   // measured on kh_2d 1024^2 (kernel ms): 8 owners + ring warpgroup 0.0595 (scheduler 0 carries three warps, the others
                       // two: the barrier waits for it), 7 + 1 0.0588 (balanced, but 1024 = 4.6 strips), 11 + 1 0.0528 (three warps per scheduler)
#endif
constexpr int NW = HX_T2D_NW;         // owner warps = 32-cell segments of the strip
// NW a multiple of 4: the ring warp gets a warpgroup of its own (three idle warps) and gives registers back (setmaxnreg).
// Otherwise the ring warp shares the last warpgroup with owners (NW + 1 a multiple of 4: every scheduler holds the same number of
// warps) and all warps keep the launch allocation.
constexpr bool REBAL = NW % 4 == 0;
static_assert(REBAL || (NW + 1) % 4 == 0, "NW or NW + 1 must be a multiple of 4");
constexpr int TXS = NW * 32;          // owner cells per strip row
constexpr int PXS = TXS + 4;          // staged row: strip + 2 ghost cells on each side
constexpr int HXS = PXS / 2;          // a TMA box is at most 256 elements wide: a row arrives as two halves of 130 cells (1040 B each),
                                      // staged as [half][field][130]
// doubles between the two halves of a staged row of nv fields (TMA destinations are 128-byte aligned)
constexpr int half_stride(int nv) { return (nv * HXS * 8 + 127) / 128 * 128 / 8; }
// offset of cell c (0 .. PXS-1) of field 0 inside a staged row of nv fields; the field stride is HXS
__device__ __forceinline__ int row_off(int c, int nv) { return c < HXS ? c : half_stride(nv) + (c - HXS); }
constexpr int NTHREADS = (REBAL ? NW + 4 : NW + 1) * 32;
constexpr int REGS_LAUNCH = (65536 / NTHREADS) / 8 * 8;   // 168 with twelve warps
#ifndef HX_T2D_REGS_RING
#define HX_T2D_REGS_RING 136   // measured on kh_2d 1024^2: 104 (spills in the ring path) 0.0705 ms, 120 0.0650, 136 0.0586, 152 0.0600, 168 0.0582
#endif
constexpr int REGS_RING = HX_T2D_REGS_RING;
constexpr int REGS_OWNER = REBAL ? (REGS_LAUNCH * (NW + 4) - REGS_RING * 4) / NW / 8 * 8 : REGS_LAUNCH;   // 184
static_assert(!REBAL || REGS_OWNER * NW + REGS_RING * 4 <= REGS_LAUNCH * (NW + 4), "setmaxnreg budgets exceed the launch allocation");

enum { GRAV_OFF = 0, GRAV_ANY = 1 };

struct Args {
  StepArgs s;
  int yc;            // rows per y chunk
  // UNI instantiations only (bitwise-uniform tables): constants of the two axes
  double uf[2];      // hw * idx (slope pre-scale), times the limiter's lim_scale
  double uhc[2];     // (dt/2) / delta_d
  double uil[2];     // 1 / delta_d
};

template <int NV>
struct Smem {
  static constexpr int NF = NV + 2;   // predicted-state record: rho, u, v, P, E, c_s, scalars
  static constexpr size_t row_bytes = (size_t)NV * PXS * sizeof(double);                 // what the two TMA copies of a row deliver
  static constexpr size_t row_stride = 2 * (size_t)half_stride(NV) * sizeof(double);
  static constexpr int NPL = 3;
  static constexpr int XN = TXS + 2;                           // x-exchange slots ex = -1 .. TXS-1 (+1 pad)
  static constexpr int XSTR = NF * XN;                         // doubles of one parity buffer
  static constexpr size_t fixed = NPL * row_stride + 2 * (size_t)XSTR * sizeof(double) + 64 + 128;
  static constexpr size_t total(int yc) { return fixed + 5 * (size_t)(yc + 6) * sizeof(double); }   // + y tables of one chunk
};

template <int NV>
__device__ __forceinline__ void tma_load_row(const CUtensorMap* tmap, double* dst, uint64_t* bar, int x, int y) {
#pragma unroll
  for (int h = 0; h < 2; ++h)
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
            smem_u32(dst + h * half_stride(NV))),
        "l"(tmap), "r"(x + h * HXS), "r"(y), "r"(0), "r"(smem_u32(bar))
        : "memory");
}

// ------------------------------------------------------------------------------------------------
// Pointwise pieces.  Field order of W / U: rho, u|m [2], P|E, scalars f|rho f.
// ------------------------------------------------------------------------------------------------
template <int NV>
__device__ __forceinline__ void prim_of_cons(const Phys& P, const double* U, double* W) {   // Eq. 1, Eq. 5
  const double ir = rcp3(U[0]);
  W[0] = U[0];
  W[1] = U[1] * ir;
  W[2] = U[2] * ir;
  const double ke2 = fma(U[2], W[2], U[1] * W[1]);
  W[3] = P.gm1 * fma(-0.5, ke2, U[3]);
#pragma unroll
  for (int s = 4; s < NV; ++s) W[s] = U[s] * ir;
}

// One face of the cell along DIR: face primitives Wc + sc t (Eq. 17), their conserved form Uf, and the analytic flux
// of that state accumulated into the half-step increment dU with the signed, (dt/2)-scaled coefficient (Eq. 18).
template <int NV, int DIR>
__device__ __forceinline__ void face_cons_flux(const Phys& P, const double* Wc, const double* t, double sc, double coef, double* Uf, double* dU) {
  double Wf[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) Wf[v] = fma(sc, t[v], Wc[v]);
  const double r = Wf[0];
  Uf[0] = r;
  Uf[1] = r * Wf[1];
  Uf[2] = r * Wf[2];
  const double ke2 = fma(Uf[2], Wf[2], Uf[1] * Wf[1]);
  Uf[3] = fma(0.5, ke2, Wf[3] * P.igm1);
  const double unc = Wf[1 + DIR] * coef;
  dU[0] = fma(r, unc, dU[0]);
  dU[1] = fma(Uf[1], unc, dU[1]);
  dU[2] = fma(Uf[2], unc, dU[2]);
  dU[1 + DIR] = fma(Wf[3], coef, dU[1 + DIR]);
  dU[3] = fma(Uf[3] + Wf[3], unc, dU[3]);
#pragma unroll
  for (int s = 4; s < NV; ++s) {
    Uf[s] = r * Wf[s];
    dU[s] = fma(Uf[s], unc, dU[s]);
  }
}

// N predicted face states U^{n+1/2} = cons(Wf) + dU (Eq. 18) as the records the Riemann solver consumes
// (q = rho, u, v, P, E, c_s, scalars f), advanced stage by stage so that the dependent chains interleave.
template <int NV, int N>
__device__ __forceinline__ void pred_states(const Phys& P, const double* const* Uf, const double* dU, double* const* q) {
  double r[N], m1[N], m2[N], E[N], mm[N], ir[N], e[N], x[N], c[N];
#pragma unroll
  for (int k = 0; k < N; ++k) {
    r[k] = Uf[k][0] + dU[0];
    m1[k] = Uf[k][1] + dU[1];
    m2[k] = Uf[k][2] + dU[2];
    E[k] = Uf[k][3] + dU[3];
  }
  rcp3_n<N>(r, ir);
#pragma unroll
  for (int k = 0; k < N; ++k) mm[k] = m1[k] * m1[k];
#pragma unroll
  for (int k = 0; k < N; ++k) mm[k] = fma(m2[k], m2[k], mm[k]);
#pragma unroll
  for (int k = 0; k < N; ++k) e[k] = fma(-0.5 * ir[k], mm[k], E[k]);
#pragma unroll
  for (int k = 0; k < N; ++k) x[k] = (P.gamma * P.gm1) * ir[k] * e[k];
  sqrt3_n<N>(x, c);
#pragma unroll
  for (int k = 0; k < N; ++k) {
    q[k][0] = r[k];
    q[k][1] = m1[k] * ir[k];
    q[k][2] = m2[k] * ir[k];
    q[k][3] = P.gm1 * e[k];
    q[k][4] = E[k];
    q[k][5] = c[k];
#pragma unroll
    for (int s = 4; s < NV; ++s) q[k][2 + s] = (Uf[k][s] + dU[s]) * ir[k];
  }
}

// HLL / HLLC flux along DIR from two records (L | R): F = rho, m[2], E, scalars.  Davis wave speeds (R14), ties per
// R15; tangential momentum and scalars ride the mass flux.
template <int NV, int RS, int DIR>
__device__ __forceinline__ void riemann_fs(const Phys& P, const double* L, const double* R, double* F) {
  constexpr int NF = NV + 2;
  const double uL = L[1 + DIR], uR = R[1 + DIR];
  const double SL = dmin(uL - L[5], uR - R[5]);
  const double SR = dmax(uL + L[5], uR + R[5]);
  const bool hllc = (RS == HX_RIEMANN_HLLC) || (RS < 0 && P.riemann == HX_RIEMANN_HLLC);
  if (hllc) {
    const double dL = SL - uL, dR = SR - uR;
    const double mL = L[0] * dL, mR = R[0] * dR;
    const double Ss = (R[3] - L[3] + uL * mL - uR * mR) * rcp3(mL - mR);
    const bool left = (SL >= 0.0) || (Ss >= 0.0);
    const bool upwind = (SL >= 0.0) || (!left && SR <= 0.0);   // pure F_L or F_R
    double qk[NF];
#pragma unroll
    for (int v = 0; v < NF; ++v) qk[v] = left ? L[v] : R[v];
    const double SK = left ? SL : SR, mK = left ? mL : mR, dK = left ? dL : dR;
    const double rK = qk[0], uK = qk[1 + DIR], pK = qk[3], EK = qk[4];
    const double w = rcp3(SK - Ss);
    const double fac = mK * w;                      // rho*_K
    const double fr = rK * uK;                      // mass flux of side K
    const double SKe = upwind ? 0.0 : SK;
    const double F0 = fma(SKe, fac - rK, fr);
    F[0] = F0;
    F[1] = F0 * qk[1];
    F[2] = F0 * qk[2];
    F[1 + DIR] = fma(SKe, fma(fac, Ss, -fr), fma(fr, uK, pK));   // normal: F_K + S_K (rho* S* - rho_K u_K)
    const double Es = fma(dK * w, EK, (Ss - uK) * fma(fac, Ss, pK * w));   // E*_K
    F[3] = fma(SKe, Es - EK, (EK + pK) * uK);
#pragma unroll
    for (int s = 4; s < NV; ++s) F[s] = F0 * qk[2 + s];
  } else {
    // HLL: (SR F_L - SL F_R + SL SR (U_R - U_L)) / (SR - SL), upwind flux outside the fan
    const bool useL = SL >= 0.0, useR = (!useL) && SR <= 0.0;
    const double iw = rcp3(SR - SL);
    const double aL = useL ? 1.0 : (useR ? 0.0 : SR * iw), aR = useL ? 0.0 : (useR ? 1.0 : -SL * iw);
    const double dd = (useL || useR) ? 0.0 : SL * SR * iw;
    const double frL = L[0] * uL, frR = R[0] * uR;
    F[0] = aL * frL + aR * frR + dd * (R[0] - L[0]);
#pragma unroll
    for (int d = 0; d < 2; ++d) {
      const double mL = L[0] * L[1 + d], mR = R[0] * R[1 + d];
      const double fL = mL * uL + (d == DIR ? L[3] : 0.0), fR = mR * uR + (d == DIR ? R[3] : 0.0);
      F[1 + d] = aL * fL + aR * fR + dd * (mR - mL);
    }
    F[3] = aL * ((L[4] + L[3]) * uL) + aR * ((R[4] + R[3]) * uR) + dd * (R[4] - L[4]);
#pragma unroll
    for (int s = 4; s < NV; ++s) {
      const double sL = L[0] * L[2 + s], sR = R[0] * R[2 + s];
      F[s] = aL * (sL * uL) + aR * (sR * uR) + dd * (sR - sL);
    }
  }
}

// The two HLLC fluxes of a cell's lower faces (x: k = 0, y: k = 1) at once, stage by stage (same arithmetic as riemann_fs)
template <int NV>
__device__ __forceinline__ void hllc_xy(const double* const* L, const double* const* R, double* const* F) {
  constexpr int NF = NV + 2, N = 2;
  double uL[N], uR[N], SL[N], SR[N], dL[N], dR[N], mL[N], mR[N], num[N], den[N], Ss[N], w[N];
#pragma unroll
  for (int k = 0; k < N; ++k) {
    uL[k] = L[k][1 + k];
    uR[k] = R[k][1 + k];
    SL[k] = dmin(uL[k] - L[k][5], uR[k] - R[k][5]);
    SR[k] = dmax(uL[k] + L[k][5], uR[k] + R[k][5]);
    dL[k] = SL[k] - uL[k];
    dR[k] = SR[k] - uR[k];
    mL[k] = L[k][0] * dL[k];
    mR[k] = R[k][0] * dR[k];
    den[k] = mL[k] - mR[k];
    num[k] = fma(-uR[k], mR[k], fma(uL[k], mL[k], R[k][3] - L[k][3]));
  }
  rcp3_n<N>(den, w);
  double qk[N][NF], SK[N], mK[N], dK[N], SKe[N], x[N];
#pragma unroll
  for (int k = 0; k < N; ++k) {
    Ss[k] = num[k] * w[k];
    const bool left = (SL[k] >= 0.0) || (Ss[k] >= 0.0);
    const bool upwind = (SL[k] >= 0.0) || (!left && SR[k] <= 0.0);
#pragma unroll
    for (int v = 0; v < NF; ++v) qk[k][v] = left ? L[k][v] : R[k][v];
    SK[k] = left ? SL[k] : SR[k];
    mK[k] = left ? mL[k] : mR[k];
    dK[k] = left ? dL[k] : dR[k];
    SKe[k] = upwind ? 0.0 : SK[k];
    x[k] = SK[k] - Ss[k];
  }
  rcp3_n<N>(x, w);
#pragma unroll
  for (int k = 0; k < N; ++k) {
    const double uK = qk[k][1 + k], pK = qk[k][3], EK = qk[k][4];
    const double fac = mK[k] * w[k];                      // rho*_K
    const double fr = qk[k][0] * uK;                      // mass flux of side K
    const double F0 = fma(SKe[k], fac - qk[k][0], fr);
    const double t1 = fma(fac, Ss[k], -fr);
    const double t3 = fma(fac, Ss[k], pK * w[k]);
    const double Es = fma(dK[k] * w[k], EK, (Ss[k] - uK) * t3);   // E*_K
    F[k][0] = F0;
    F[k][1] = F0 * qk[k][1];
    F[k][2] = F0 * qk[k][2];
    F[k][1 + k] = fma(SKe[k], t1, fma(fr, uK, pK));
    F[k][3] = fma(SKe[k], Es - EK, (EK + pK) * uK);
#pragma unroll
    for (int s = 4; s < NV; ++s) F[k][s] = F0 * qk[k][2 + s];
  }
}

// ------------------------------------------------------------------------------------------------
// The kernel.  Warps 0..NW-1 own the cells ex = 32 warp + lane of the strip; lanes 0 and 1 of warp NW handle the ring
// cells ex = -1 (provides its predicted x+ state) and ex = TXS (solves the x face on its left); warps NW+1..NW+3
// only complete the ring warpgroup for setmaxnreg and leave.
// ------------------------------------------------------------------------------------------------
template <int NV, int GRAV, int LIM, int RS, bool UNI>
__global__ void __launch_bounds__(NTHREADS, 1) step_tile2d_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ Args a) {
  using SM = Smem<NV>;
  constexpr int NF = SM::NF, XN = SM::XN;
  constexpr int PSTR = (int)(SM::row_stride / sizeof(double));
  extern __shared__ unsigned char smem_raw[];
  unsigned char* base = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
  double* rows = (double*)base;
  double* const X0 = (double*)(base + SM::NPL * SM::row_stride);   // parity buffer 0; buffer 1 follows
  uint64_t* mbar = (uint64_t*)(X0 + 2 * SM::XSTR);
  double* yt = (double*)(mbar + 8);   // y-axis tables of this chunk

  const StepArgs& s = a.s;
  const Layout& L = s.L;
  const Tables& T = s.T;
  const Phys& P = s.P;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const bool owner = wid < NW;
  constexpr int NSYNC = (NW + 1) * 32;   // threads at the per-row barrier (id 1): the owners and the ring warp

  const int i0 = blockIdx.x * TXS;
  const int k0 = blockIdx.y * a.yc, k1 = min(L.n[1], k0 + a.yc);
  const int ex = owner ? (wid * 32 + lane) : (lane == 0 ? -1 : TXS);
  const bool act = owner || (wid == NW && lane < 2);
  const int xoff = owner ? 0 : (lane == 0 ? -1 : 1);        // ring: the second ghost layer cell this thread converts too
  const int i = i0 + ex;
  const bool st_ok = owner && i < L.n[0];
  const int cidx = row_off(ex + 2, NV);                       // offset of the own cell inside field 0 of a staged row (field stride HXS)
  const int cim = row_off(ex + 1, NV), cip = row_off(ex + 3, NV);   // ... of its x neighbours
  const int xs_own = ex + 1, xs_nbr = ex;
  const bool lim_none = (LIM == HX_LIM_NONE) || (LIM < 0 && P.limiter == HX_LIM_NONE);   // R19: no predictor

  // ---- loop-invariant geometry of this column, (dt/2) folded in ------------------------------------
  const double hdt = 0.5 * s.dt;
  const int pi = min(max(i + NG, 1), L.np[0] - 2);
  double flx, fhx, hc0, il0;
  if (UNI) {
    flx = fhx = a.uf[0];
    hc0 = a.uhc[0];
    il0 = a.uil[0];
  } else {
    const double hwx = T.hw[0][pi];
    flx = hwx * T.idx[0][pi];
    fhx = hwx * T.idx[0][pi + 1];
    hc0 = hdt * T.cf[0][0][0][pi];     // Cartesian: dS/dV of both x faces = 1 / width
    il0 = T.lf[0][0][pi];
  }
  const double k0c = 2.0 * hc0;
  const double hgx = (GRAV == GRAV_ANY) ? hdt * T.grav[0][pi] : 0.0;

  // ---- TMA prologue: rows k0-2, k0-1, k0 -----------------------------------------------------------------
  const int xs = i0 + L.lead;                                 // box origin in storage coordinates (cell i0-2)
  uint32_t phase = 0u;
  if (threadIdx.x == 0) {
    mbar_init(&mbar[0], 1);
    mbar_init(&mbar[1], 1);
    mbar_init(&mbar[2], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  const int yb = max(k0 - 3 + NG, 0), ylen = a.yc + 6;
  for (int q = threadIdx.x; q < ylen; q += blockDim.x) {
    const int py = min(yb + q, L.np[1] - 1);
    yt[q] = T.hw[1][py];
    yt[ylen + q] = T.idx[1][py];
    yt[2 * ylen + q] = T.cf[1][0][1][py];
    yt[3 * ylen + q] = T.grav[1][py];
    yt[4 * ylen + q] = T.lf[1][1][py];
  }
  auto YT = [&](int k, int py) { return yt[k * ylen + (py - yb)]; };
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int b = 0; b < 3; ++b) {
      mbar_expect_tx(&mbar[b], (uint32_t)SM::row_bytes);
      tma_load_row<NV>(&tmap, rows + b * PSTR, &mbar[b], xs, k0 - 2 + b + NG);
    }
  }

  auto convert = [&](double* rw, int off, double* Wout, bool store) {
    double U[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) U[v] = rw[v * HXS + off];
    prim_of_cons<NV>(P, U, Wout);
    if (store) {
#pragma unroll
      for (int v = 0; v < NV; ++v) rw[v * HXS + off] = Wout[v];
    }
  };
  auto convert_row = [&](double* rw, double* Wown) {
    convert(rw, cidx, Wown, act);
    if (xoff != 0 && act) {
      double tmp[NV];
      convert(rw, row_off(ex + 2 + xoff, NV), tmp, true);
    }
  };

  double dym[NV];             // W(p) - W(p-1) of this column
  {
    double Wm2[NV], Wc0[NV];
    mbar_wait(&mbar[0], 0u);
    convert(rows, cidx, Wm2, false);
    mbar_wait(&mbar[1], 0u);
    phase = 3u;
    convert_row(rows + PSTR, Wc0);
#pragma unroll
    for (int v = 0; v < NV; ++v) dym[v] = Wc0[v] - Wm2[v];
    __syncthreads();          // everyone has read row k0-2: its buffer takes row k0+1
    if (threadIdx.x == 0) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(&mbar[0], (uint32_t)SM::row_bytes);
      tma_load_row<NV>(&tmap, rows, &mbar[0], xs, k0 + 1 + NG);
    }
  }
  // register rebalancing, one setmaxnreg per warpgroup: the ring warpgroup gives registers back, the owners take them
  if (REBAL) {
    if (owner) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REGS_OWNER));
    else asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REGS_RING));
  }
  if (wid > NW) {             // the rest of the ring warpgroup was only needed for setmaxnreg: wait in the final reduction
    block_rate_max(0.0, s.rate_bits);
    return;
  }

  double yp[NF];              // predicted state on the upper y face of the previous row
  double Up[NV];              // partially updated cell of the previous row
  double Un0 = 0.0, Unm[2] = {0.0, 0.0};   // rho^n, m^n of the previous row (time-centred gravity)
  double Ul[4] = {1.0, 0.0, 0.0, 1.0};     // rho, m, E of the cell written one iteration ago (deferred CFL rate)
  bool st_l = false;
  double rate_max = 0.0;
  bool bad = false;
#pragma unroll
  for (int v = 0; v < NF; ++v) yp[v] = 1.0;
#pragma unroll
  for (int v = 0; v < NV; ++v) Up[v] = 1.0;
  double* outp = s.Uout + L.off(min(i, L.n[0] - 1) + NG, k0 - 2 + NG, 0);   // cell (i, p-1) at p = k0-1

  // A7: CFL rate + positivity check of the cell in Ul (padded row index pyc), one iteration after it was written
  auto cfl_rate = [&](int pyc) {
    const double mm = fma(Ul[2], Ul[2], Ul[1] * Ul[1]);
    const double ir = rcp3(Ul[0]);
    const double e = fma(-0.5 * ir, mm, Ul[3]);
    const double cs = sqrt3((P.gamma * P.gm1) * ir * e);     // e <= 0 (or rho, e of opposite sign) gives NaN
    const double il1 = UNI ? a.uil[1] : YT(4, max(pyc, yb));
    const double rate = fma(fma(fabs(Ul[1]), ir, cs), il0, fma(fabs(Ul[2]), ir, cs) * il1);
    const bool fine = (Ul[0] > 0.0) && (rate < __longlong_as_double(0x7ff0000000000000LL));
    rate_max = (st_l && fine && rate > rate_max) ? rate : rate_max;
    bad = bad || (st_l && !fine);
  };

  // O2-O4 for the cell of row p: limited slopes, the four face states, half-step increment dU (Eq. 17-18, unsplit)
  auto predictor = [&](const double* Pc, const double* Wn, int py, double* Wc, double* dU, double* Uxm, double* Uxp, double* Uym, double* Uyp,
                       double& hc1) {
    double fly, fhy;
    if (UNI) {
      fly = fhy = a.uf[1];
      hc1 = a.uhc[1];
    } else {
      const double hwy = YT(0, py);
      fly = hwy * YT(1, py);
      fhy = hwy * YT(1, py + 1);
      hc1 = hdt * YT(2, py);
    }
    double t[NV], dm[NV], dp[NV];   // (runtime-switch builds: all slopes of a direction behind one branch on the limiter)
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      Wc[v] = Pc[v * HXS + cidx];
      dU[v] = 0.0;
      const double wm = Pc[v * HXS + cim], wp = Pc[v * HXS + cip];
      dm[v] = Wc[v] - wm;
      dp[v] = wp - Wc[v];
      if constexpr (LIM >= 0) t[v] = lim_pre<LIM, UNI>(P.limiter, dm[v], dp[v], flx, fhx);
    }
    if constexpr (LIM < 0) lim_pre_n<NV, LIM, UNI>(P.limiter, dm, dp, &flx, &fhx, t);
    face_cons_flux<NV, 0>(P, Wc, t, UNI ? -flx : -lim_scale<LIM>(), hc0, Uxm, dU);
    face_cons_flux<NV, 0>(P, Wc, t, UNI ? flx : lim_scale<LIM>(), -hc0, Uxp, dU);
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      dp[v] = Wn[v] - Wc[v];
      if constexpr (LIM >= 0) t[v] = lim_pre<LIM, UNI>(P.limiter, dym[v], dp[v], fly, fhy);
    }
    if constexpr (LIM < 0) lim_pre_n<NV, LIM, UNI>(P.limiter, dym, dp, &fly, &fhy, t);
#pragma unroll
    for (int v = 0; v < NV; ++v) dym[v] = dp[v];
    face_cons_flux<NV, 1>(P, Wc, t, UNI ? -fly : -lim_scale<LIM>(), hc1, Uym, dU);
    face_cons_flux<NV, 1>(P, Wc, t, UNI ? fly : lim_scale<LIM>(), -hc1, Uyp, dU);
    if (GRAV == GRAV_ANY) {   // half step of rho g, m . g (R13)
      const double rho = Wc[0], hgy = hdt * YT(3, py);
      dU[1] = fma(rho, hgx, dU[1]);
      dU[2] = fma(rho, hgy, dU[2]);
      dU[3] = fma(rho * Wc[1], hgx, fma(rho * Wc[2], hgy, dU[3]));
    }
    if (lim_none) {
#pragma unroll
      for (int v = 0; v < NV; ++v) dU[v] = 0.0;
    }
  };

  constexpr bool HLLC_STATIC = (RS == HX_RIEMANN_HLLC);
  auto march = [&](auto own_tag) {
    constexpr bool OWN = decltype(own_tag)::value;
    int bc = 1;                 // buffer of row p
    int xo = 0;                 // offset of this row's exchange buffer (toggles between the two parity buffers)
#pragma unroll 1
    for (int p = k0 - 1; p <= k1; ++p, outp += L.sy) {
      const int py = p + NG;
      const int bn = (bc == 2) ? 0 : bc + 1;
      double* Pc = rows + bc * PSTR;
      double* Pn = rows + bn * PSTR;
      double* const X = X0 + xo;                           // exchange slots of this row ...
      double* const Xo = X0 + (SM::XSTR - xo);             // ... and of the previous row (fluxes through its upper x faces)
      xo = SM::XSTR - xo;
      mbar_wait(&mbar[bn], (phase >> bn) & 1u);            // row p+1 has arrived (issued a whole iteration ago)
      phase ^= (1u << bn);
      double Wn[NV], Wc[NV], dU[NV], hc1;
      double Uf[4][NV];          // conserved face states: 0 x-, 1 x+, 2 y-, 3 y+
      if constexpr (OWN) {
        // ======== block 1: slopes, half-step increment, the four predicted states, the deferred CFL rate of cell p-2
        cfl_rate(py - 2);
        convert(Pn, cidx, Wn, true);                       // cons -> prim of the own cell of row p+1, in place
        predictor(Pc, Wn, py, Wc, dU, Uf[0], Uf[1], Uf[2], Uf[3], hc1);
        double qxm[NF], qym[NF], ypn[NF];
        {
          double qa[NF];
          const double* const ua[2] = {Uf[1], Uf[2]};
          double* const qo[2] = {qa, qym};
          pred_states<NV, 2>(P, ua, dU, qo);
#pragma unroll
          for (int v = 0; v < NF; ++v) X[v * XN + xs_own] = qa[v];
        }
        {
          const double* const ub[2] = {Uf[0], Uf[3]};
          double* const qo[2] = {qxm, ypn};
          pred_states<NV, 2>(P, ub, dU, qo);
        }
        double Un[NV];           // U^n of cell p
        {
          const double rho = Wc[0];
          Un[0] = rho;
          Un[1] = rho * Wc[1];
          Un[2] = rho * Wc[2];
          Un[3] = fma(0.5, fma(Un[2], Wc[2], Un[1] * Wc[1]), Wc[3] * P.igm1);
#pragma unroll
          for (int sv = 4; sv < NV; ++sv) Un[sv] = rho * Wc[sv];
        }
        asm volatile("bar.sync 1, %0;" ::"n"(NSYNC) : "memory");   // x+ states visible; all reads of row p done; last row's fluxes visible
        if (threadIdx.x == 0 && p + 3 <= k1 + 1) {           // row p+3 takes the buffer of row p
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          mbar_expect_tx(&mbar[bc], (uint32_t)SM::row_bytes);
          tma_load_row<NV>(&tmap, Pc, &mbar[bc], xs, p + 3 + NG);
        }
        // ======== block 2: the flux through the upper x face of cell p-1 comes back in its own slot; the two Riemann
        // problems on the lower faces of cell p (the x flux goes back into the neighbour's slot); finish cell p-1 with
        // the y flux, start cell p
#pragma unroll
        for (int v = 0; v < NV; ++v) Up[v] = fma(-k0c, Xo[v * XN + xs_own], Up[v]);
        double Fx[NV], Fy[NV];
        {
          double qlx[NF];
#pragma unroll
          for (int v = 0; v < NF; ++v) qlx[v] = X[v * XN + xs_nbr];
          if (HLLC_STATIC || (RS < 0 && P.riemann == HX_RIEMANN_HLLC)) {
            const double* const Ls[2] = {qlx, yp};
            const double* const Rs[2] = {qxm, qym};
            double* const Fs[2] = {Fx, Fy};
            hllc_xy<NV>(Ls, Rs, Fs);
          } else {
            riemann_fs<NV, RS, 0>(P, qlx, qxm, Fx);
            riemann_fs<NV, RS, 1>(P, yp, qym, Fy);
          }
#pragma unroll
          for (int v = 0; v < NV; ++v) X[v * XN + xs_nbr] = Fx[v];
        }
#pragma unroll
        for (int v = 0; v < NF; ++v) yp[v] = ypn[v];
        {   // the flux through the upper y face of cell p-1 is Fy: write the cell once
          const double k1p = UNI ? 2.0 * a.uhc[1] : 2.0 * hdt * YT(2, py - 1);
          double Unew[NV];
#pragma unroll
          for (int v = 0; v < NV; ++v) Unew[v] = fma(-k1p, Fy[v], Up[v]);
          if (GRAV == GRAV_ANY) {   // time-centred (R13)
            const double hgyp = hdt * YT(3, py - 1);
            const double rs = Un0 + Unew[0];
            const double m1 = fma(rs, hgx, Unew[1]), m2 = fma(rs, hgyp, Unew[2]);
            Unew[3] = fma(Unm[0] + m1, hgx, fma(Unm[1] + m2, hgyp, Unew[3]));
            Unew[1] = m1;
            Unew[2] = m2;
          }
          st_l = st_ok && (p > k0);
          if (st_l) {
#pragma unroll
            for (int v = 0; v < NV; ++v) outp[v * L.sv] = Unew[v];
          }
#pragma unroll
          for (int v = 0; v < 4; ++v) Ul[v] = Unew[v];
        }
        {   // cell p: U^n + the two lower faces
          const double k1m = 2.0 * hc1;
#pragma unroll
          for (int v = 0; v < NV; ++v) Up[v] = fma(k1m, Fy[v], fma(k0c, Fx[v], Un[v]));
          if (GRAV == GRAV_ANY) {
            Un0 = Un[0];
            Unm[0] = Un[1];
            Unm[1] = Un[2];
          }
        }
      } else {
        // ======== ring warp (lanes 0, 1): predictor, one predicted state, at most one Riemann solve ================
        convert_row(Pn, Wn);
        predictor(Pc, Wn, py, Wc, dU, Uf[0], Uf[1], Uf[2], Uf[3], hc1);
        double q[NF];
        {
          double Usel[NV];      // left ring cell: its x+ face; right ring cell: its x- face
#pragma unroll
          for (int v = 0; v < NV; ++v) Usel[v] = (lane == 0) ? Uf[1][v] : Uf[0][v];
          const double* const us[1] = {Usel};
          double* const qo[1] = {q};
          pred_states<NV, 1>(P, us, dU, qo);
        }
        if (lane == 0) {
#pragma unroll
          for (int v = 0; v < NF; ++v) X[v * XN + xs_own] = q[v];
        }
        asm volatile("bar.sync 1, %0;" ::"n"(NSYNC) : "memory");
        if (lane == 1) {
          double ql[NF], F[NV];
#pragma unroll
          for (int v = 0; v < NF; ++v) ql[v] = X[v * XN + xs_nbr];
          riemann_fs<NV, RS, 0>(P, ql, q, F);
#pragma unroll
          for (int v = 0; v < NV; ++v) X[v * XN + xs_nbr] = F[v];
        }
      }
      bc = bn;
    }
  };
  if (owner) {
    march(std::true_type{});
    cfl_rate(k1 + 1 + NG - 2);                             // the last cell written (row k1-1)
  } else {
    march(std::false_type{});
  }
  if (bad) atomicOr(s.status, 1);
  block_rate_max(rate_max, s.rate_bits);
}

}  // namespace t2d
}  // namespace hx

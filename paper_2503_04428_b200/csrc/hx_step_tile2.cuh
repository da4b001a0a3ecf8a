// hx_step_tile2.cuh -- the fused 3-D step kernel (A1-A7 of SURVEY 8(a) in ONE pass over HBM), second design.
//
// Why a second design: ncu on the first tiled kernel (profiles/r1a_*) showed the FP64 pipe only half busy with
// the issue port just as loaded (fp64 : other instructions = 1 : 1), 22 % of the threads doing full work on ring
// cells, and 3 warps per scheduler.  This kernel
//   * owns a 32 x 8 tile per CTA (warp <-> row, lane <-> cell) and marches along z; the one-cell ring around the
//     tile is handled by FOUR extra warps (bottom row, top row, left column, right column) that run only what the
//     tile needs from them (slopes, half-step increment, one predicted face state, at most one Riemann solve);
//   * rebalances the register file with setmaxnreg: the ring warpgroup gives registers back, the two owner
//     warpgroups take them, because ptxas interleaves the owners' independent fp64 chains only with ~190 registers;
//   * exchanges every neighbour quantity through shared memory: slope neighbours are read from the staged
//     primitive plane; the predicted "+" face state of a cell goes into the cell's own exchange slot, the
//     neighbour across that face reads it, solves the Riemann problem once and writes the flux back INTO THE
//     SAME SLOT, where the first cell picks it up as the flux through its upper face;
//   * stages planes (tile + 2 ghost layers, all fields) with one TMA bulk-tensor copy each into a 3-deep ring,
//     and the z-axis tables of the chunk once;
//   * keeps the owner iteration straight-line (no edge-iteration branches), batches the predicted states and the
//     three HLLC solves stage by stage, defers the CFL rate of a cell by one plane, and advances passive scalars
//     one at a time after the hydro fields (register peak);
//   * trims the arithmetic: reciprocal / square root = MUFU seed + one cubic correction, limiters on pre-scaled
//     one-sided differences, flux differences accumulated straight into the half-step increment, tangential
//     momentum and scalar fluxes as (value x mass flux);
//   * keeps geometry out of registers on bitwise-uniform Cartesian grids (UNI: kernel-parameter constants), and
//     as per-thread / per-plane 1-D table products otherwise;
//   * is instantiated for the ideal gas (Eq. 5) and, for nvar 9, for the gas + radiation EOS (Eq. 6-7, Newton-
//     Raphson for T inside the kernel); one instantiation carries the internal-energy monitoring of Eq. 10-12 (EMON).
//
// PAPER.md: Eq. 17 (slopes), Eq. 18 + Toro 16.5 (unsplit predictor), Eq. 19 (update), L201 (HLL/HLLC),
// Eq. 13-16 (spherical sources), Eq. 2-4 (gravity), Eq. 5-7 (EOS), Eq. 10-12 (monitoring); readings R1-R29.
#pragma once
#include <cuda.h>

#include <type_traits>

#include "hx_common.cuh"

namespace hx {
namespace t2 {

constexpr int TX = 32;        // owner cells per tile row = one warp
constexpr int PX = TX + 4;    // staged plane row: tile + 2 ghost cells on each side (36 * 8 B = 18 * 16 B)
#ifndef HX_T2_TY
#define HX_T2_TY 8
#endif
constexpr int TY_DEFAULT = HX_T2_TY;   // 8 owner rows (two warpgroups) + 4 ring warps (one warpgroup): two owner warps and one ring warp per scheduler

// Register budgets after setmaxnreg.  The pool is what the CTA was given at launch, (TY+4) warps x 32 x REGS_LAUNCH
// (not the whole 64 K file): the owners' increase must fit into what the ring warpgroup releases, or
// setmaxnreg.inc waits forever.
// Measured (A/B on B200): ring 96..120 is equal for the Cartesian builds (96 with twelve owner rows).  The spherical ring path used to need 136
// (nine fields at once, per-thread geometry products); with the scalars advanced one at a time (RING2) and the geometry
// read from the shared column / row tables it runs in 120 like the Cartesian one from eight fields on (wedge_3d, nvar 9:
// 104 -> 7.78 ms, 120 -> 7.31, 136 -> 7.51); the nvar 5-7 spherical builds keep 136 (sedov_wedge_3d: 1.14 vs 1.18 ms).
#ifndef HX_T2_REGS_RING_SPH
#define HX_T2_REGS_RING_SPH 120
#endif
#ifdef HX_T2_REGS_RING
constexpr int ring_regs(bool, int, int = TY_DEFAULT) { return HX_T2_REGS_RING; }
#else
constexpr int ring_regs(bool sph, int nv, int ty = TY_DEFAULT) { return ty > 8 ? 96 : ((sph && nv < 8) ? 136 : (sph ? HX_T2_REGS_RING_SPH : 120)); }
#endif
constexpr int regs_launch(int ty) { return (65536 / ((ty + 4) * 32)) / 8 * 8; }
constexpr int owner_regs(bool sph, int nv, int ty = TY_DEFAULT) {
  const int raw = (regs_launch(ty) * (ty + 4) - ring_regs(sph, nv, ty) * 4) / ty / 8 * 8;
  return raw > 232 ? 232 : raw;
}
static_assert(owner_regs(true, 5) * TY_DEFAULT + ring_regs(true, 5) * 4 <= regs_launch(TY_DEFAULT) * (TY_DEFAULT + 4), "setmaxnreg budgets exceed the launch allocation");
static_assert(owner_regs(true, 9) * TY_DEFAULT + ring_regs(true, 9) * 4 <= regs_launch(TY_DEFAULT) * (TY_DEFAULT + 4), "setmaxnreg budgets exceed the launch allocation");
static_assert(owner_regs(false, 5) * TY_DEFAULT + ring_regs(false, 5) * 4 <= regs_launch(TY_DEFAULT) * (TY_DEFAULT + 4), "setmaxnreg budgets exceed the launch allocation");
static_assert(owner_regs(false, 5, 12) * 12 + ring_regs(false, 5, 12) * 4 <= regs_launch(12) * 16, "setmaxnreg budgets exceed the launch allocation");

constexpr bool writes_x_ghosts(bool uni, int ty) { return uni && ty == 8; }   // builds whose boundary threads also write the x-ghost cells

enum { GRAV_OFF = 0, GRAV_ANY = 1, GRAV_Z = 2, GRAV_R = 3 };   // GRAV_Z / GRAV_R: acceleration along direction 2 / 0 only (uniform g along z; point mass, self-gravity)
constexpr bool grav_has(int grav, int d, bool sph = false) {
  return (grav == GRAV_ANY && !(sph && d == 2)) || (grav == GRAV_Z && d == 2) || (grav == GRAV_R && d == 0);   // spherical builds: never along phi
}

struct Args {
  StepArgs s;
  int zc;            // planes per z chunk
  int bcx_lo, bcx_hi; // boundary conditions of direction 0: the owners of the first / last two cells of a row also write the x-ghost
                      // images of their cells (A0 for direction 0 folded into the update: the data is in registers, and x-ghost
                      // columns are the expensive part of a separate fill -- one 64-byte DRAM burst per 16 useful bytes)
  // UNI instantiations only (bitwise-uniform Cartesian tables): constants of the three axes
  double uf[3];      // hw * idx   (slope pre-scale, = 1/2 up to rounding), times lim_scale of a build with a static limiter (1/2 for MC)
  double uhc[3];     // (dt/2) / delta_d
  double uil[3];     // 1 / delta_d  (CFL inverse lengths)
};

// One CTA-wide barrier per plane instead of two: the exchange slots are double buffered by plane parity, so the flux a
// neighbour writes back into a slot during plane p is picked up after the barrier of plane p+1 while the "+" states
// of plane p+1 already sit in the other buffer.  Needs twice the slot memory: field counts whose buffers fit.
#ifndef HX_T2_RING2_NV
#define HX_T2_RING2_NV 8
#endif
#ifndef HX_T2_UNROLL
#define HX_T2_UNROLL 1
#endif
#ifndef HX_T2_ONEBAR
#define HX_T2_ONEBAR 1
#endif
#ifndef HX_T2_ONEBAR_NV
#define HX_T2_ONEBAR_NV 8    // nvar 9 would fit with two z chunks, but their overhead eats the gain (wedge_3d 7.317 -> 7.303 ms, wedge_3d_rad 13.69 -> 13.97)
#endif
constexpr bool one_barrier(int nv) { return HX_T2_ONEBAR && nv <= HX_T2_ONEBAR_NV; }

template <int NV, int TY>
struct Smem {
  static constexpr bool ONEBAR = one_barrier(NV);
  static constexpr int NXY = ONEBAR ? 2 : 1;
  static constexpr int PY = TY + 4;
  static constexpr int NF = NV + 2;
  static constexpr int FSTR = PY * PX;                         // field stride inside a plane (doubles)
  static constexpr size_t plane_bytes = (size_t)NV * FSTR * sizeof(double);
  static constexpr size_t plane_stride = (plane_bytes + 127) / 128 * 128;
  static constexpr int NPL = 3;
  static constexpr int XP = TX + 1;                            // x-exchange row pitch: slots ex = -1 .. TX-1 (odd pitch: conflict-free columns)
  static constexpr int XSTR = TY * XP;                         // field stride of the x-exchange buffer
  static constexpr int YSTR = (TY + 1) * TX;                   // y-exchange: slots ey = -1 .. TY-1
  static constexpr size_t x_bytes = (size_t)NF * XSTR * sizeof(double);
  static constexpr size_t y_bytes = (size_t)NF * YSTR * sizeof(double);
  // nvar >= 8: the passive-scalar parts of the four predicted states an owner keeps across the first barrier go to
  // private shared-memory slots instead of registers (the nvar-9 builds spilled them to local memory: long-scoreboard stalls)
  static constexpr int NPRIV = (NV >= 8) ? 4 * (NV - 5) : 0;
  static constexpr size_t priv_bytes = (size_t)NPRIV * TY * TX * sizeof(double);
  // spherical builds: 1-D factors of the slope, predictor, update and CFL coefficients by tile column and tile row
  // (15 + 12 tables), read (and multiplied) at use, so that the ~27 loop-invariant per-thread products need no
  // registers (they used to be spilled to local memory, which the 16 KB of L1 left beside the tile cannot hold)
  static constexpr int GT_X = TX + 2, GT_Y = TY + 2, NGX = 15, NGY = 12, GT_N = NGX * GT_X + NGY * GT_Y;
  static constexpr int XYSTR = NF * (XSTR + YSTR);             // doubles of one parity buffer (X fields, then Y fields)
  static constexpr size_t fixed = NPL * plane_stride + NXY * (x_bytes + y_bytes) + priv_bytes + 64 + 128;
  // + the column / row factor tables (spherical builds) + the z tables of one chunk: hw, idx, dS-/dV, dS+/dV, g, 1/l along z;
  // in spherical geometry dS-/dV, dS+/dV and 1/l are one and the same table (1 / dphi), stored once, and there is no
  // acceleration along phi (uniform gravity on a spherical grid runs on the generic kernel)
  static constexpr int nzt(bool sph) { return sph ? 3 : 6; }
  static constexpr size_t total(int zc, bool sph) { return fixed + (sph ? GT_N * sizeof(double) : 0) + nzt(sph) * (size_t)(zc + 6) * sizeof(double); }
};

// ------------------------------------------------------------------------------------------------
// fp64 helpers.  rcp.approx / rsqrt.approx give ~20 good bits (the low input word is ignored); one
// cubic correction brings the relative error to ~(2^-19)^3 = 2^-57, below one ulp.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double rcp3(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y, 1.0);
  const double t = fma(e, e, e);
  return fma(y, t, y);
}

__device__ __forceinline__ double sqrt3(double x) {   // x > 0
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double t = x * y;                       // ~ sqrt(x) (1 + d)
  const double e = fma(-t, y, 1.0);             // 1 - x y^2
  const double q = fma(0.375, e, 0.5) * e;      // (1 - e)^(-1/2) - 1 = e/2 + 3 e^2/8 + O(e^3)
  return fma(t, q, t);
}

// scale the caller applies to what lim_core returns
template <int LIM>
__device__ __forceinline__ constexpr double lim_scale() { return LIM == HX_LIM_MC ? 0.5 : 1.0; }

__device__ __forceinline__ int hi32(double x) { return __double2hiint(x); }
// plain compare-select minimum / maximum (no NaN quieting: inputs are finite wherever the result is used)
__device__ __forceinline__ double dmin(double a, double b) { return (a < b) ? a : b; }
__device__ __forceinline__ double dmax(double a, double b) { return (a > b) ? a : b; }
// true when a and b have opposite sign bits
__device__ __forceinline__ bool opp_sign(double a, double b) { return ((hi32(a) ^ hi32(b)) & 0x80000000) != 0; }

// limiter on one-sided differences a (backward), b (forward); all are homogeneous of degree 1
template <int LIM>
__device__ __forceinline__ double lim_core(int lim_rt, double a, double b) {
  if (LIM == HX_LIM_MINMOD) {
    const bool opp = opp_sign(a, b);
    const double r = (fabs(a) < fabs(b)) ? a : b;
    return opp ? 0.0 : r;
  }
  if (LIM == HX_LIM_MC) {   // returns TWICE the limited value (the caller's face scale carries the 1/2): saves a multiply
    const bool opp = opp_sign(a, b);
    const double sum = a + b;
    const double m = (fabs(a) < fabs(b)) ? a : b;
    const double m4 = 4.0 * m;
    const double r = (fabs(m4) < fabs(sum)) ? m4 : sum;   // 2 min(2|a|, 2|b|, |a+b|/2) with the common sign
    return opp ? 0.0 : r;
  }
  // van Leer 2ab/(a+b), van Albada ab(a+b)/(a^2+b^2) (R4), zero across extrema; the runtime-switch build (LIM < 0)
  // dispatches here on a warp-uniform value.  Reciprocals by seed + cubic correction instead of IEEE division.
  const int lim = LIM < 0 ? lim_rt : LIM;
  if (lim == HX_LIM_NONE) return 0.0;
  if (lim == HX_LIM_MINMOD) return lim_core<HX_LIM_MINMOD>(lim_rt, a, b);
  if (lim == HX_LIM_MC) return 0.5 * lim_core<HX_LIM_MC>(lim_rt, a, b);
  const double ab = a * b;
  double r;
  if (lim == HX_LIM_VANLEER) r = 2.0 * ab * rcp3(a + b);
  else r = ab * (a + b) * rcp3(fma(a, a, b * b));
  return (ab > 0.0) ? r : 0.0;
}

// hw * lim(dm * idx_lo, dp * idx_hi)  (Eq. 17 with R5); fl = hw*idx_lo, fh = hw*idx_hi.  On uniform grids
// (fl == fh) the common factor is left to the caller, who folds it into the face-state FMA.
template <int LIM, bool UNI>
__device__ __forceinline__ double lim_pre(int lim_rt, double dm, double dp, double fl, double fh) {
  if (LIM == HX_LIM_NONE) return 0.0;
  if (UNI) return lim_core<LIM>(lim_rt, dm, dp);
  return lim_core<LIM>(lim_rt, dm * fl, dp * fh);
}

// N limited slopes at once: the runtime-switch builds (LIM < 0) branch ONCE on the warp-uniform limiter for all N
// instead of once per slope (21-33 slopes per cell: the branches cost instructions and keep ptxas from interleaving the
// slopes' chains).  fl / fh: one pre-scale pair for all (PER = false) or one per slope (PER = true).
template <int N, int LIM, bool UNI, bool PER = false>
__device__ __forceinline__ void lim_pre_n(int lim_rt, const double* dm, const double* dp, const double* fl, const double* fh, double* t) {
  if (LIM >= 0) {
#pragma unroll
    for (int v = 0; v < N; ++v) t[v] = lim_pre<LIM, UNI>(lim_rt, dm[v], dp[v], fl[PER ? v : 0], fh[PER ? v : 0]);
    return;
  }
  double a[N], b[N];
#pragma unroll
  for (int v = 0; v < N; ++v) {   // uniform grids: the common factor is left to the caller's face-state FMA (as in lim_pre)
    a[v] = UNI ? dm[v] : dm[v] * fl[PER ? v : 0];
    b[v] = UNI ? dp[v] : dp[v] * fh[PER ? v : 0];
  }
  switch (lim_rt) {
    case HX_LIM_MINMOD:
#pragma unroll
      for (int v = 0; v < N; ++v) t[v] = lim_core<HX_LIM_MINMOD>(0, a[v], b[v]);
      break;
    case HX_LIM_MC:
#pragma unroll
      for (int v = 0; v < N; ++v) t[v] = 0.5 * lim_core<HX_LIM_MC>(0, a[v], b[v]);
      break;
    case HX_LIM_VANLEER:
#pragma unroll
      for (int v = 0; v < N; ++v) t[v] = lim_core<HX_LIM_VANLEER>(0, a[v], b[v]);
      break;
    case HX_LIM_VANALBADA:
#pragma unroll
      for (int v = 0; v < N; ++v) t[v] = lim_core<HX_LIM_VANALBADA>(0, a[v], b[v]);
      break;
    default:
#pragma unroll
      for (int v = 0; v < N; ++v) t[v] = 0.0;
  }
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
      "T2_WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra.uni T2_WAIT_DONE;\n"
      "bra.uni T2_WAIT_LOOP;\n"
      "T2_WAIT_DONE:\n"
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

// ------------------------------------------------------------------------------------------------
// Gas + radiation EOS (Eq. 6-7; EOS == HX_EOS_GAS_RADIATION instantiations).  T is the positive root of
// a1 T + a4 T^4 = b, by Newton-Raphson as the paper prescribes (L102), from the smaller single-term root (the
// iterate then only moves down), until the correction is a few ulp (R27); reciprocals by seed + cubic correction.
// ------------------------------------------------------------------------------------------------
// Tg > 0: start from this guess instead (the temperature of the cell centre for its face and predicted states: a
// start below the root overshoots once and then descends like any other; 2-3 steps instead of 6-8, same root).
__device__ __forceinline__ double gr_temperature(double a1, double a4, double b, double Tg = 0.0) {
  // non-physical (e <= 0 or P <= 0): NaN -> P, c_s and the CFL rate are NaN and the rate check reports it (a negative T
  // would give a POSITIVE radiation-dominated pressure a_r T^4 / 3 again)
  if (!(b > 0.0)) return __longlong_as_double(0x7ff8000000000000LL);
  double T = (Tg > 0.0) ? Tg : dmin(b * rcp3(a1), sqrt3(sqrt3(b * rcp3(a4))));
  for (int it = 0; it < 60; ++it) {
    const double T3 = T * T * T;
    const double step = (fma(a4 * T3, T, a1 * T) - b) * rcp3(fma(4.0 * a4, T3, a1));
    T -= step;
    if (fabs(step) <= 1e-15 * T) break;
  }
  return T;
}
// P and c_s from (rho, 1/rho, e); e from (rho, P)
__device__ __forceinline__ void gr_from_energy(const Phys& P, double rho, double ir, double e, double& p, double& c, double Tg = 0.0, double* Tout = nullptr) {
  const double T = gr_temperature(rho * P.rgas * P.igm1, P.arad, e, Tg);
  if (Tout) *Tout = T;
  const double T3 = T * T * T;
  const double pg = rho * P.rgas * T;
  p = fma(P.arad * (1.0 / 3.0) * T3, T, pg);
  const double al = P.arad * (1.0 / 3.0) * T3 * ir * rcp3(P.rgas);   // P_r / P_g
  c = sqrt3(fma(al, fma(16.0, al, 20.0), P.gamma * P.igm1) * rcp3(fma(12.0, al, P.igm1)) * P.rgas * T);
}
__device__ __forceinline__ double gr_energy_of_T(const Phys& P, double rho, double T) {   // Eq. 6a
  const double T2 = T * T;
  return fma(P.arad, T2 * T2, rho * P.rgas * T * P.igm1);
}
__device__ __forceinline__ double gr_energy(const Phys& P, double rho, double p, double Tg = 0.0, double* Tout = nullptr) {
  const double T = gr_temperature(rho * P.rgas, P.arad * (1.0 / 3.0), p, Tg);
  if (Tout) *Tout = T;
  const double T2 = T * T;
  return fma(P.arad, T2 * T2, rho * P.rgas * T * P.igm1);
}

template <int N>
__device__ __forceinline__ void gr_from_energy_n(const Phys& P, const double* rho, const double* ir, const double* e, double* p, double* c, double Tg,
                                                 double* Tout = nullptr);
template <int N>
__device__ __forceinline__ void gr_energy_n(const Phys& P, const double* rho, const double* p, double Tg, double* e);

// ------------------------------------------------------------------------------------------------
// Pointwise pieces of the scheme.  Field order of W / U: rho, u|m [3], P|E, scalars f|rho f.
// ------------------------------------------------------------------------------------------------
// gas + radiation EOS: coll = all 32 lanes of the warp are here together (the fast solve is warp-collective); Tg = a nearby
// temperature to start it from; Tout: the temperature found
template <int NV, int EOS = HX_EOS_IDEAL>
__device__ __forceinline__ void prim_of_cons(const Phys& P, const double* U, double* W, bool coll = false, double Tg = 0.0, double* Tout = nullptr) {   // Eq. 1, Eq. 5 / 6
  const double ir = rcp3(U[0]);
  W[0] = U[0];
  W[1] = U[1] * ir;
  W[2] = U[2] * ir;
  W[3] = U[3] * ir;
  const double ke2 = fma(U[3], W[3], fma(U[2], W[2], U[1] * W[1]));
  if (EOS == HX_EOS_IDEAL) {
    W[4] = P.gm1 * fma(-0.5, ke2, U[4]);
  } else {
    double c;
    const double e = fma(-0.5, ke2, U[4]);
    if (coll) gr_from_energy_n<1>(P, &U[0], &ir, &e, &W[4], &c, Tg, Tout);   // warp-collective: coll must be warp-uniform
    else gr_from_energy(P, U[0], ir, e, W[4], c, Tg, Tout);   // Newton loop, from the guess when it is positive
  }
#pragma unroll
  for (int s = 5; s < NV; ++s) W[s] = U[s] * ir;
}

// One face of the cell along DIR: face primitives Wc + sc t (Eq. 17; sc = -+1, or -+hw*idx on uniform grids), their conserved form Uf, and the
// analytic flux of that state accumulated into the half-step increment dU with the signed, (dt/2)-scaled
// area/volume coefficient `coef` (Eq. 18: + for the lower face, - for the upper face).
template <int NV, int DIR, int EOS = HX_EOS_IDEAL>
__device__ __forceinline__ void face_cons_flux(const Phys& P, const double* Wc, const double* t, double sc, double coef, double* Uf, double* dU,
                                               double* unc_out = nullptr, double* pf_out = nullptr) {
  // gas + radiation EOS: the internal energy e(rho_f, P_f) of the face state is left out here (Uf[4] and the energy flux);
  // the caller solves for the six of a cell at once and adds them (pf_out: the face pressure it needs for that)
  double Wf[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) Wf[v] = fma(sc, t[v], Wc[v]);
  const double r = Wf[0];
  Uf[0] = r;
  Uf[1] = r * Wf[1];
  Uf[2] = r * Wf[2];
  Uf[3] = r * Wf[3];
  const double ke2 = fma(Uf[3], Wf[3], fma(Uf[2], Wf[2], Uf[1] * Wf[1]));
  Uf[4] = (EOS == HX_EOS_IDEAL) ? fma(0.5, ke2, Wf[4] * P.igm1) : 0.5 * ke2;
  if (EOS != HX_EOS_IDEAL && pf_out) *pf_out = Wf[4];
  const double unc = Wf[1 + DIR] * coef;
  if (unc_out) *unc_out = unc;   // signed (dt/2) dS/dV u_n of this face: what a passive scalar's flux rides on
  dU[0] = fma(r, unc, dU[0]);
  dU[1] = fma(Uf[1], unc, dU[1]);
  dU[2] = fma(Uf[2], unc, dU[2]);
  dU[3] = fma(Uf[3], unc, dU[3]);
  dU[1 + DIR] = fma(Wf[4], coef, dU[1 + DIR]);
  dU[4] = fma(Uf[4] + Wf[4], unc, dU[4]);
#pragma unroll
  for (int s = 5; s < NV; ++s) {
    Uf[s] = r * Wf[s];
    dU[s] = fma(Uf[s], unc, dU[s]);
  }
}

// Predicted face state U^{n+1/2} = cons(Wf) + dU (Eq. 18) as the record the Riemann solver consumes:
// q = rho, u[3], P, E, c_s, scalars f.
template <int NV, int EOS = HX_EOS_IDEAL>
__device__ __forceinline__ void pred_state(const Phys& P, const double* Uf, const double* dU, double* q, double Tg = 0.0) {
  const double r = Uf[0] + dU[0];
  const double m1 = Uf[1] + dU[1], m2 = Uf[2] + dU[2], m3 = Uf[3] + dU[3];
  const double E = Uf[4] + dU[4];
  const double mm = fma(m3, m3, fma(m2, m2, m1 * m1));   // independent of 1/rho: shortens the dependent chain
  const double ir = rcp3(r);
  const double e = fma(-0.5 * ir, mm, E);                // internal energy density
  q[0] = r;
  q[1] = m1 * ir;
  q[2] = m2 * ir;
  q[3] = m3 * ir;
  q[5] = E;
  if (EOS == HX_EOS_IDEAL) {
    q[4] = P.gm1 * e;
    q[6] = sqrt3((P.gamma * P.gm1) * ir * e);            // c^2 = gamma P / rho
  } else {
    gr_from_energy(P, r, ir, e, q[4], q[6], Tg);
  }
#pragma unroll
  for (int s = 5; s < NV; ++s) q[2 + s] = (Uf[s] + dU[s]) * ir;
}

// HLL / HLLC flux along DIR from two records (L | R): F = rho, m[3], E, scalars.  Davis wave speeds
// (R14), ties per R15.  Tangential momenta and scalars ride the mass flux: F_K + S_K (U*_K - U_K)
// = q_K (rho_K u_K + S_K (rho*_K - rho_K)) for every quantity advected with the contact.
template <int NV, int RS, int DIR>
__device__ __forceinline__ void riemann_fs(const Phys& P, const double* L, const double* R, double* F) {
  constexpr int NF = NV + 2;
  const double uL = L[1 + DIR], uR = R[1 + DIR];
  const double SL = dmin(uL - L[6], uR - R[6]);
  const double SR = dmax(uL + L[6], uR + R[6]);
  const bool hllc = (RS == HX_RIEMANN_HLLC) || (RS < 0 && P.riemann == HX_RIEMANN_HLLC);
  if (hllc) {
    const double dL = SL - uL, dR = SR - uR;
    const double mL = L[0] * dL, mR = R[0] * dR;
    const double Ss = (R[4] - L[4] + uL * mL - uR * mR) * rcp3(mL - mR);
    const bool left = (SL >= 0.0) || (Ss >= 0.0);
    const bool upwind = (SL >= 0.0) || (!left && SR <= 0.0);   // pure F_L or F_R
    double qk[NF];
#pragma unroll
    for (int v = 0; v < NF; ++v) qk[v] = left ? L[v] : R[v];
    const double SK = left ? SL : SR, mK = left ? mL : mR, dK = left ? dL : dR;
    const double rK = qk[0], uK = qk[1 + DIR], pK = qk[4], EK = qk[5];
    const double w = rcp3(SK - Ss);
    const double fac = mK * w;                      // rho*_K
    const double fr = rK * uK;                      // mass flux of side K
    const double SKe = upwind ? 0.0 : SK;
    const double F0 = fma(SKe, fac - rK, fr);
    F[0] = F0;
    F[1] = F0 * qk[1];
    F[2] = F0 * qk[2];
    F[3] = F0 * qk[3];
    F[1 + DIR] = fma(SKe, fma(fac, Ss, -fr), fma(fr, uK, pK));   // normal: F_K + S_K (rho* S* - rho_K u_K)
    const double Es = fma(dK * w, EK, (Ss - uK) * fma(fac, Ss, pK * w));   // E*_K
    F[4] = fma(SKe, Es - EK, (EK + pK) * uK);
#pragma unroll
    for (int s = 5; s < NV; ++s) F[s] = F0 * qk[2 + s];
  } else {
    // HLL: (SR F_L - SL F_R + SL SR (U_R - U_L)) / (SR - SL), upwind flux outside the fan
    const bool useL = SL >= 0.0, useR = (!useL) && SR <= 0.0;
    const double iw = rcp3(SR - SL);
    const double aL = useL ? 1.0 : (useR ? 0.0 : SR * iw), aR = useL ? 0.0 : (useR ? 1.0 : -SL * iw);
    const double dd = (useL || useR) ? 0.0 : SL * SR * iw;
    const double frL = L[0] * uL, frR = R[0] * uR;
    F[0] = aL * frL + aR * frR + dd * (R[0] - L[0]);
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const double mL = L[0] * L[1 + d], mR = R[0] * R[1 + d];
      const double fL = mL * uL + (d == DIR ? L[4] : 0.0), fR = mR * uR + (d == DIR ? R[4] : 0.0);
      F[1 + d] = aL * fL + aR * fR + dd * (mR - mL);
    }
    F[4] = aL * ((L[5] + L[4]) * uL) + aR * ((R[5] + R[4]) * uR) + dd * (R[5] - L[5]);
#pragma unroll
    for (int s = 5; s < NV; ++s) {
      const double sL = L[0] * L[2 + s], sR = R[0] * R[2 + s];
      F[s] = aL * (sL * uL) + aR * (sR * uR) + dd * (sR - sL);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Batched forms: N independent instances advanced stage by stage, so that the instruction stream handed
// to ptxas already interleaves the dependent chains (1/x and sqrt seeds + corrections, S*, fluxes).  ncu
// showed ptxas emitting the sequential calls as sequential chains (every DFMA waiting its full latency).
// ------------------------------------------------------------------------------------------------
template <int N>
__device__ __forceinline__ void rcp3_n(const double* x, double* y) {
  double s[N], e[N];
#pragma unroll
  for (int k = 0; k < N; ++k) asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(s[k]) : "d"(x[k]));
#pragma unroll
  for (int k = 0; k < N; ++k) e[k] = fma(-x[k], s[k], 1.0);
#pragma unroll
  for (int k = 0; k < N; ++k) e[k] = fma(e[k], e[k], e[k]);
#pragma unroll
  for (int k = 0; k < N; ++k) y[k] = fma(s[k], e[k], s[k]);
}

template <int N>
__device__ __forceinline__ void sqrt3_n(const double* x, double* y) {
  double s[N], t[N], e[N];
#pragma unroll
  for (int k = 0; k < N; ++k) asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(s[k]) : "d"(x[k]));
#pragma unroll
  for (int k = 0; k < N; ++k) t[k] = x[k] * s[k];
#pragma unroll
  for (int k = 0; k < N; ++k) e[k] = fma(-t[k], s[k], 1.0);
#pragma unroll
  for (int k = 0; k < N; ++k) s[k] = fma(0.375, e[k], 0.5);
#pragma unroll
  for (int k = 0; k < N; ++k) e[k] = s[k] * e[k];
#pragma unroll
  for (int k = 0; k < N; ++k) y[k] = fma(t[k], e[k], t[k]);
}

// N roots of a1 T + a4 T^4 = b at once, from the guess Tg > 0 (the temperature of a neighbouring state: the cell centre for
// its face and predicted states, the cell below for a cell centre, the old time level for the new state).  Halley steps
// (cubic convergence, f'' = 12 a4 T^2) advanced stage by stage for all N so that their dependent chains interleave, until
// every instance in the warp has a correction below 2e-6 T -- the iterate after it is then converged to ~1e-17 (relative
// error e -> 1.25 e^3) -- at most four; an instance that is not there yet (a strong shock, a non-physical input) goes
// through the Newton loop.  f is increasing and convex for T > 0: the root is unique, so this is the oracle's root to
// rounding (R27).  WARP-COLLECTIVE (the early exit is a warp vote): all 32 lanes must call it together, whatever their data;
// a lane whose guess is not positive (first plane, garbage beyond the domain edge) takes the Newton loop afterwards.
template <int N>
__device__ __forceinline__ void gr_temperature_n(const double* a1, double a4, const double* b, double Tg, double* T) {
  double t[N], s[N];
  const bool guess = Tg > 0.0;                          // per lane; a lane without a usable guess idles through the collective part
#pragma unroll
  for (int k = 0; k < N; ++k) t[k] = guess ? Tg : 1.0;
  const double a46 = 6.0 * a4;
#pragma unroll 1
  for (int it = 0; it < 4; ++it) {
    double T2[N], q[N], f[N], fp[N], den[N], r[N];
#pragma unroll
    for (int k = 0; k < N; ++k) T2[k] = t[k] * t[k];
#pragma unroll
    for (int k = 0; k < N; ++k) q[k] = a4 * T2[k] * t[k];
#pragma unroll
    for (int k = 0; k < N; ++k) f[k] = fma(q[k], t[k], fma(a1[k], t[k], -b[k]));
#pragma unroll
    for (int k = 0; k < N; ++k) fp[k] = fma(4.0, q[k], a1[k]);
#pragma unroll
    for (int k = 0; k < N; ++k) den[k] = fma(fp[k], fp[k], -(f[k] * (a46 * T2[k])));
    rcp3_n<N>(den, r);
#pragma unroll
    for (int k = 0; k < N; ++k) s[k] = f[k] * fp[k] * r[k];
#pragma unroll
    for (int k = 0; k < N; ++k) t[k] -= s[k];
    bool ok = true;
#pragma unroll
    for (int k = 0; k < N; ++k) ok = ok && (fabs(s[k]) <= 2e-6 * t[k]);
    if (__all_sync(0xffffffffu, ok || !guess)) break;
  }
#pragma unroll
  for (int k = 0; k < N; ++k) {
    T[k] = t[k];
    if (!(guess && (b[k] > 0.0) && (fabs(s[k]) <= 2e-6 * t[k]))) T[k] = gr_temperature(a1[k], a4, b[k], (guess && t[k] > 0.0) ? t[k] : 0.0);
  }
}

// P and c_s of N states from (rho, 1/rho, e) (Eq. 6b, Eq. 7); e of N states from (rho, P) (Eq. 6a)
template <int N>
__device__ __forceinline__ void gr_from_energy_n(const Phys& P, const double* rho, const double* ir, const double* e, double* p, double* c, double Tg,
                                                 double* Tout) {
  double a1[N], T[N], pr3[N], al[N], x[N], y[N], w[N];
#pragma unroll
  for (int k = 0; k < N; ++k) a1[k] = rho[k] * P.rgas * P.igm1;
  gr_temperature_n<N>(a1, P.arad, e, Tg, T);
  const double ar3 = P.arad * (1.0 / 3.0), irg = rcp3(P.rgas);
#pragma unroll
  for (int k = 0; k < N; ++k) pr3[k] = ar3 * (T[k] * T[k] * T[k]);
#pragma unroll
  for (int k = 0; k < N; ++k) {
    p[k] = fma(pr3[k], T[k], rho[k] * P.rgas * T[k]);
    al[k] = pr3[k] * ir[k] * irg;                                   // P_r / P_g
    x[k] = fma(12.0, al[k], P.igm1);
    if (Tout) Tout[k] = T[k];
  }
  rcp3_n<N>(x, w);
#pragma unroll
  for (int k = 0; k < N; ++k) y[k] = fma(al[k], fma(16.0, al[k], 20.0), P.gamma * P.igm1) * w[k] * P.rgas * T[k];
  sqrt3_n<N>(y, c);
}
template <int N>
__device__ __forceinline__ void gr_energy_n(const Phys& P, const double* rho, const double* p, double Tg, double* e) {
  double a1[N], T[N];
#pragma unroll
  for (int k = 0; k < N; ++k) a1[k] = rho[k] * P.rgas;
  gr_temperature_n<N>(a1, P.arad * (1.0 / 3.0), p, Tg, T);
#pragma unroll
  for (int k = 0; k < N; ++k) e[k] = gr_energy_of_T(P, rho[k], T[k]);
}

// N predicted face states at once (same arithmetic as pred_state)
template <int NV, int N, int EOS = HX_EOS_IDEAL>
__device__ __forceinline__ void pred_states(const Phys& P, const double* const* Uf, const double* dU, double* const* q, double* const* ir_out = nullptr, double Tg = 0.0) {
  double r[N], m1[N], m2[N], m3[N], E[N], mm[N], ir[N], e[N], x[N], c[N];
#pragma unroll
  for (int k = 0; k < N; ++k) {
    r[k] = Uf[k][0] + dU[0];
    m1[k] = Uf[k][1] + dU[1];
    m2[k] = Uf[k][2] + dU[2];
    m3[k] = Uf[k][3] + dU[3];
    E[k] = Uf[k][4] + dU[4];
  }
  rcp3_n<N>(r, ir);
#pragma unroll
  for (int k = 0; k < N; ++k) mm[k] = m1[k] * m1[k];
#pragma unroll
  for (int k = 0; k < N; ++k) mm[k] = fma(m2[k], m2[k], mm[k]);
#pragma unroll
  for (int k = 0; k < N; ++k) mm[k] = fma(m3[k], m3[k], mm[k]);
#pragma unroll
  for (int k = 0; k < N; ++k) e[k] = fma(-0.5 * ir[k], mm[k], E[k]);
  double pr[N];
  if (EOS == HX_EOS_IDEAL) {
#pragma unroll
    for (int k = 0; k < N; ++k) x[k] = (P.gamma * P.gm1) * ir[k] * e[k];
    sqrt3_n<N>(x, c);
#pragma unroll
    for (int k = 0; k < N; ++k) pr[k] = P.gm1 * e[k];
  } else {
    gr_from_energy_n<N>(P, r, ir, e, pr, c, Tg);
  }
#pragma unroll
  for (int k = 0; k < N; ++k) {
    q[k][0] = r[k];
    q[k][1] = m1[k] * ir[k];
    q[k][2] = m2[k] * ir[k];
    q[k][3] = m3[k] * ir[k];
    q[k][4] = pr[k];
    q[k][5] = E[k];
    q[k][6] = c[k];
    if (ir_out) *ir_out[k] = ir[k];
#pragma unroll
    for (int s = 5; s < NV; ++s) q[k][2 + s] = (Uf[k][s] + dU[s]) * ir[k];
  }
}

// N HLLC fluxes at once; instance k is the face normal to direction dir[k] (same arithmetic as riemann_fs)
template <int NV, int N>
__device__ __forceinline__ void hllc_n(const int (&dir)[N], const double* const* L, const double* const* R, double* const* F) {
  constexpr int NF = NV + 2;
  double uL[N], uR[N], SL[N], SR[N], dL[N], dR[N], mL[N], mR[N], num[N], den[N], Ss[N], w[N];
#pragma unroll
  for (int k = 0; k < N; ++k) {
    uL[k] = L[k][1 + dir[k]];
    uR[k] = R[k][1 + dir[k]];
    SL[k] = dmin(uL[k] - L[k][6], uR[k] - R[k][6]);
    SR[k] = dmax(uL[k] + L[k][6], uR[k] + R[k][6]);
  }
#pragma unroll
  for (int k = 0; k < N; ++k) {
    dL[k] = SL[k] - uL[k];
    dR[k] = SR[k] - uR[k];
  }
#pragma unroll
  for (int k = 0; k < N; ++k) {
    mL[k] = L[k][0] * dL[k];
    mR[k] = R[k][0] * dR[k];
  }
#pragma unroll
  for (int k = 0; k < N; ++k) {
    den[k] = mL[k] - mR[k];
    num[k] = fma(-uR[k], mR[k], fma(uL[k], mL[k], R[k][4] - L[k][4]));
  }
  rcp3_n<N>(den, w);
#pragma unroll
  for (int k = 0; k < N; ++k) Ss[k] = num[k] * w[k];
  double qk[N][NF], SK[N], mK[N], dK[N], SKe[N], x[N];
#pragma unroll
  for (int k = 0; k < N; ++k) {
    const bool left = (SL[k] >= 0.0) || (Ss[k] >= 0.0);
    const bool upwind = (SL[k] >= 0.0) || (!left && SR[k] <= 0.0);   // pure F_L or F_R
#pragma unroll
    for (int v = 0; v < NF; ++v) qk[k][v] = left ? L[k][v] : R[k][v];
    SK[k] = left ? SL[k] : SR[k];
    mK[k] = left ? mL[k] : mR[k];
    dK[k] = left ? dL[k] : dR[k];
    SKe[k] = upwind ? 0.0 : SK[k];
    x[k] = SK[k] - Ss[k];
  }
  rcp3_n<N>(x, w);
  double fac[N], fr[N], F0[N], t1[N], t2[N], t3[N], Es[N];
#pragma unroll
  for (int k = 0; k < N; ++k) {
    fac[k] = mK[k] * w[k];                               // rho*_K
    fr[k] = qk[k][0] * qk[k][1 + dir[k]];                 // mass flux of side K
    t3[k] = qk[k][4] * w[k];
    t2[k] = dK[k] * w[k];
  }
#pragma unroll
  for (int k = 0; k < N; ++k) {
    F0[k] = fma(SKe[k], fac[k] - qk[k][0], fr[k]);
    t1[k] = fma(fac[k], Ss[k], -fr[k]);
    t3[k] = fma(fac[k], Ss[k], t3[k]);
  }
#pragma unroll
  for (int k = 0; k < N; ++k) {
    const double uK = qk[k][1 + dir[k]], pK = qk[k][4], EK = qk[k][5];
    Es[k] = fma(t2[k], EK, (Ss[k] - uK) * t3[k]);         // E*_K
    F[k][0] = F0[k];
    F[k][1] = F0[k] * qk[k][1];
    F[k][2] = F0[k] * qk[k][2];
    F[k][3] = F0[k] * qk[k][3];
    F[k][1 + dir[k]] = fma(SKe[k], t1[k], fma(fr[k], uK, pK));   // normal: F_K + S_K (rho* S* - rho_K u_K)
    F[k][4] = fma(SKe[k], Es[k] - EK, (EK + pK) * uK);
#pragma unroll
    for (int s = 5; s < NV; ++s) F[k][s] = F0[k] * qk[k][2 + s];
  }
}

// Internal-energy monitoring (Eq. 10-12, R29; EMON instantiations): per face, from the two records and the
// mass flux of the Riemann solution, the advective flux of e (mass flux x e/rho of the upwind state) and the face
// velocity (contact speed S*, or u_L / u_R when the fan lies on one side).
template <int DIR>
__device__ __forceinline__ void monitor_rec(const double* L, const double* R, double fmass, double& phi, double& uf) {
  const double uL = L[1 + DIR], uR = R[1 + DIR];
  const double SL = dmin(uL - L[6], uR - R[6]), SR = dmax(uL + L[6], uR + R[6]);
  const double mL = L[0] * (SL - uL), mR = R[0] * (SR - uR);
  const double Ss = (R[4] - L[4] + uL * mL - uR * mR) * rcp3(mL - mR);
  uf = (SL >= 0.0) ? uL : ((SR <= 0.0) ? uR : Ss);
  const bool left = fmass >= 0.0;
  const double r = left ? L[0] : R[0], E = left ? L[5] : R[5];
  const double u1 = left ? L[1] : R[1], u2 = left ? L[2] : R[2], u3 = left ? L[3] : R[3];
  phi = fmass * fma(-0.5 * r, fma(u3, u3, fma(u2, u2, u1 * u1)), E) * rcp3(r);
}

__device__ __forceinline__ double monitor_blend2(double eps, double en, double e1, double e2, double ek) {   // Eq. 11-12
  const double lim = eps * ek;
  double alpha;
  if (e1 >= lim) alpha = 1.0;
  else if (e1 > 0.1 * lim) alpha = (e1 * rcp3(lim)) * (e1 * rcp3(lim));
  else alpha = 0.0;
  return en + alpha * (e1 - en) + (1.0 - alpha) * (e2 - en);
}

// ------------------------------------------------------------------------------------------------
// The kernel.  Thread roles (warp-uniform except in the last warp):
//   warps 0..TY-1  owners of row ey = warp, cell ex = lane
//   warp  TY       bottom ring row  ey = -1   -> provides the predicted y+ state of its cells
//   warp  TY+1     top ring row     ey = TY   -> solves the y face below it
//   warp  TY+2     left ring column  ex = -1  (lanes 0..TY-1)  -> provides the predicted x+ state
//   warp  TY+3     right ring column ex = TX  (lanes 0..TY-1)  -> solves the x face on its left
// The owner warps and the ring warps form separate warpgroups and rebalance the register file with
// setmaxnreg: the ring path needs far fewer registers than it is given at launch, and ptxas interleaves the
// independent fp64 chains of the owner path only when it has ~200 registers (at 168 it emits them serially).
// ------------------------------------------------------------------------------------------------
template <int NV, bool SPH, int GRAV, int LIM, int RS, bool UNI, int TY, int EOS = HX_EOS_IDEAL, bool EMON = false>
__global__ void __launch_bounds__((TY + 4) * 32, 1)
step_tile2_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ Args a) {
  static_assert(TY % 4 == 0 && TY >= 4 && TY <= 32, "owner warps must fill whole warpgroups (setmaxnreg)");
  static_assert(!(UNI && SPH), "UNI is for Cartesian grids");
  static_assert(EOS == HX_EOS_IDEAL || EOS == HX_EOS_GAS_RADIATION, "unknown equation of state");
  using SM = Smem<NV, TY>;
  constexpr int NF = SM::NF, FSTR = SM::FSTR, XSTR = SM::XSTR, YSTR = SM::YSTR, XP = SM::XP;
  constexpr int PSTR = (int)(SM::plane_stride / sizeof(double));
  // column / row factor tables instead of per-thread products (spherical builds): frees ~50 registers per thread
  constexpr bool GTAB = SPH;
  constexpr bool GTABP = SPH && NV >= 8;   // ... also the slope / predictor coefficients: pays from eight fields on (below, -1.4 % on the nvar-5 wedge)
  extern __shared__ unsigned char smem_raw[];
  unsigned char* base = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
  double* planes = (double*)base;
  constexpr bool ONEBAR = SM::ONEBAR;
  constexpr bool RING2 = NV >= HX_T2_RING2_NV;   // ring warps: hydro fields first, then the passive scalars one at a time
  double* const XY0 = (double*)(base + SM::NPL * SM::plane_stride);   // parity buffer 0: X fields, then Y fields; buffer 1 follows (ONEBAR)
  uint64_t* mbar = (uint64_t*)(XY0 + SM::NXY * SM::XYSTR);
  double* priv = (double*)(mbar + 8) + min((int)threadIdx.x, TY * TX - 1);   // private slots of the owner threads, field stride TY*TX
  double* gtab = (double*)(mbar + 8) + SM::NPRIV * TY * TX;   // spherical builds: column / row factor tables
  double* zt = gtab + (SPH ? SM::GT_N : 0);   // z-axis tables of this chunk, staged once (per-plane global loads stall the march)

  const StepArgs& s = a.s;
  const Layout& L = s.L;
  const Tables& T = s.T;
  const Phys& P = s.P;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const bool owner = wid < TY;
  int ex, ey, xoff = 0, coff = 0;     // tile coordinates; extra cells this thread converts (offsets from its own)
  bool act = true;
  if (owner) {
    ex = lane;
    ey = wid;
  } else if (wid == TY) {
    ex = lane;
    ey = -1;
    xoff = -PX;
    coff = (lane == 0) ? -1 : (lane == 31 ? 1 : 0);
  } else if (wid == TY + 1) {
    ex = lane;
    ey = TY;
    xoff = PX;
    coff = (lane == 0) ? -1 : (lane == 31 ? 1 : 0);
  } else {
    const bool right = wid == TY + 3;
    ex = right ? TX : -1;
    ey = min(lane, TY - 1);
    act = lane < TY;
    xoff = right ? 1 : -1;
  }

  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
  const int k0 = blockIdx.z * a.zc, k1 = min(L.n[2], k0 + a.zc);
  const int i = i0 + ex, j = j0 + ey;                       // interior indices of this thread's column
  const bool st_ok = owner && i < L.n[0] && j < L.n[1];
  // x-ghost images written by the boundary threads: only where the owner path has registers to spare -- the constant-geometry
  // eight-row builds (rt_3d +1.9 %, cold_stream_3d +2.0 % whole step; the spherical builds lose 3-5 % in the kernel, the twelve-row
  // build gains nothing: there the separate fill does it)
  constexpr bool XG = writes_x_ghosts(UNI, TY);
  const bool xedge = XG && st_ok && (i < NG || i >= L.n[0] - NG);
  const int cidx = (ey + 2) * PX + (ex + 2);                // offset of the own cell inside one field of a plane
  const int xs_own = ey * XP + ex + 1, xs_nbr = ey * XP + ex;
  const int ys_own = (ey + 1) * TX + ex, ys_nbr = ey * TX + ex;
  const bool lim_none = (LIM == HX_LIM_NONE) || (LIM < 0 && P.limiter == HX_LIM_NONE);   // R19: no predictor

  // ---- loop-invariant geometry of this column, (dt/2) folded in -----------------------------------
  const double hdt = 0.5 * s.dt;
  const int pi = min(max(i + NG, 1), L.np[0] - 2), pj = min(max(j + NG, 1), L.np[1] - 2);
  double flx, fhx, fly, fhy, hcm0, hcp0, hcm1, hcp1, c2m, c2p, il0, il1, il2xy;
  if (UNI) {
    flx = fhx = a.uf[0];
    fly = fhy = a.uf[1];
    hcm0 = hcp0 = a.uhc[0];
    hcm1 = hcp1 = a.uhc[1];
    c2m = c2p = a.uhc[2];
    il0 = a.uil[0];
    il1 = a.uil[1];
    il2xy = a.uil[2];
  } else {
    const double hwx = T.hw[0][pi], hwy = T.hw[1][pj];
    flx = hwx * T.idx[0][pi];
    fhx = hwx * T.idx[0][pi + 1];
    fly = hwy * T.idx[1][pj];
    fhy = hwy * T.idx[1][pj + 1];
    hcm0 = hdt * (T.cf[0][0][0][pi] * T.cf[0][0][1][pj]);
    hcp0 = hdt * (T.cf[0][1][0][pi] * T.cf[0][1][1][pj]);
    hcm1 = hdt * (T.cf[1][0][0][pi] * T.cf[1][0][1][pj]);
    hcp1 = hdt * (T.cf[1][1][0][pi] * T.cf[1][1][1][pj]);
    c2m = hdt * (T.cf[2][0][0][pi] * T.cf[2][0][1][pj]);
    c2p = hdt * (T.cf[2][1][0][pi] * T.cf[2][1][1][pj]);
    il0 = T.lf[0][0][pi] * T.lf[0][1][pj];
    il1 = T.lf[1][0][pi] * T.lf[1][1][pj];
    il2xy = T.lf[2][0][pi] * T.lf[2][1][pj];
  }
  // update coefficients dt dS/dV of the x and y faces; in spherical geometry the angular components
  // carry the (1 -+ rr), (1 -+ st) factors of Eq. 14 (angular-momentum conserving form)
  const double k0m = 2.0 * hcm0, k0p = 2.0 * hcp0, k1m = 2.0 * hcm1, k1p = 2.0 * hcp1;
  double kxm = k0m, kxp = k0p, kym = k1m, kyp = k1p, hgr = 0.0, hAr = 0.0, hcgt = 0.0, hcAt = 0.0;
  if (SPH) {
    const double rr = T.rr[pi], st = T.st[pj], crg = T.cr[pi];
    kxm = k0m * (1.0 - rr);
    kxp = k0p * (1.0 + rr);
    kym = k1m * (1.0 - st);
    kyp = k1p * (1.0 + st);
    hgr = hdt * T.gr[pi];
    hAr = hdt * T.Ar[pi];
    hcgt = hdt * crg * T.gt[pj];
    hcAt = hdt * crg * T.At[pj];
  }
  const double hgx = grav_has(GRAV, 0) ? hdt * T.grav[0][pi] : 0.0;
  const double hgy = grav_has(GRAV, 1) ? hdt * T.grav[1][pj] : 0.0;

  // ---- TMA prologue: planes k0-2, k0-1, k0 -------------------------------------------------------------
  const int xs = i0 + L.lead, ys = j0;                      // box origin in storage coordinates (cell i0-2, j0-2)
  uint32_t phase = 0u;
  if (threadIdx.x == 0) {
    mbar_init(&mbar[0], 1);
    mbar_init(&mbar[1], 1);
    mbar_init(&mbar[2], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // padded z indices touched by this chunk: k0-3+NG (deferred CFL rate of the first iteration, unused) .. k1+1+NG
  const int zb = max(k0 - 3 + NG, 0), zlen = a.zc + 6;
  for (int q = threadIdx.x; q < zlen; q += blockDim.x) {
    const int pz = min(zb + q, L.np[2] - 1);
    zt[q] = T.hw[2][pz];
    zt[zlen + q] = T.idx[2][pz];
    zt[2 * zlen + q] = T.cf[2][0][2][pz];
    if (!SPH) {   // spherical: cf[2][1][2] and lf[2][2] are the same table as cf[2][0][2] (1 / dphi); no acceleration along phi
      zt[3 * zlen + q] = T.grav[2][pz];
      zt[4 * zlen + q] = T.cf[2][1][2][pz];
      zt[5 * zlen + q] = T.lf[2][2][pz];
    }
  }
  if (GTAB) {   // column factors (with the (1 -+ rr) of Eq. 14) and row factors (with (1 -+ st)), (dt/2) folded in
    for (int e = threadIdx.x; e < SM::GT_X; e += blockDim.x) {
      const int pe = min(max(i0 + e - 1 + NG, 1), L.np[0] - 2);
      const double km = 2.0 * hdt * T.cf[0][0][0][pe], kp = 2.0 * hdt * T.cf[0][1][0][pe], rr = T.rr[pe], hwx = T.hw[0][pe];
      double* g = gtab + e;
      g[0 * SM::GT_X] = km;
      g[1 * SM::GT_X] = kp;
      g[2 * SM::GT_X] = km * (1.0 - rr);
      g[3 * SM::GT_X] = kp * (1.0 + rr);
      g[4 * SM::GT_X] = 2.0 * hdt * T.cr[pe];
      g[5 * SM::GT_X] = T.lf[0][0][pe];
      g[6 * SM::GT_X] = T.lf[1][0][pe];
      g[7 * SM::GT_X] = hwx * T.idx[0][pe];                 // flx
      g[8 * SM::GT_X] = hwx * T.idx[0][pe + 1];             // fhx
      g[9 * SM::GT_X] = hdt * T.cf[0][0][0][pe];            // hcm0
      g[10 * SM::GT_X] = hdt * T.cf[0][1][0][pe];           // hcp0
      g[11 * SM::GT_X] = hdt * T.cr[pe];                    // (dt/2) x the radial factor of the theta / phi face coefficients
      g[12 * SM::GT_X] = hdt * T.gr[pe];                    // hgr
      g[13 * SM::GT_X] = hdt * T.Ar[pe];                    // hAr
      g[14 * SM::GT_X] = hdt * T.grav[0][pe];               // hgx
    }
    double* gy = gtab + SM::NGX * SM::GT_X;
    for (int e = threadIdx.x; e < SM::GT_Y; e += blockDim.x) {
      const int pe = min(max(j0 + e - 1 + NG, 1), L.np[1] - 2);
      const double bm = T.cf[1][0][1][pe], bp = T.cf[1][1][1][pe], st = T.st[pe], hwy = T.hw[1][pe];
      double* g = gy + e;
      g[0 * SM::GT_Y] = bm;
      g[1 * SM::GT_Y] = bp;
      g[2 * SM::GT_Y] = bm * (1.0 - st);
      g[3 * SM::GT_Y] = bp * (1.0 + st);
      g[4 * SM::GT_Y] = T.cf[2][1][1][pe];
      g[5 * SM::GT_Y] = T.lf[1][1][pe];
      g[6 * SM::GT_Y] = T.lf[2][1][pe];
      g[7 * SM::GT_Y] = hwy * T.idx[1][pe];                 // fly
      g[8 * SM::GT_Y] = hwy * T.idx[1][pe + 1];             // fhy
      g[9 * SM::GT_Y] = T.gt[pe];
      g[10 * SM::GT_Y] = T.At[pe];
      g[11 * SM::GT_Y] = hdt * T.grav[1][pe];               // hgy
    }
  }
  // table k of the list above at padded z index pz (k: 0 hw, 1 idx, 2 dS-/dV, 3 dS+/dV, 4 g, 5 1/l)
  auto ZT = [&](int k, int pz) {
    const int slot = SPH ? (k >= 2 ? 2 : k) : (k == 3 ? 4 : (k == 4 ? 3 : k));
    return zt[slot * zlen + (pz - zb)];
  };
  auto GX = [&](int k) { return gtab[k * SM::GT_X + ex + 1]; };                       // column factor k of this thread's cell
  auto GY = [&](int k) { return gtab[SM::NGX * SM::GT_X + k * SM::GT_Y + ey + 1]; };   // row factor k
  // the loop-invariant coefficients of this thread's column: table reads at use (GTAB) or the registers set up above
  auto FLX = [&]() { return GTABP ? GX(7) : flx; };
  auto FHX = [&]() { return GTABP ? GX(8) : fhx; };
  auto FLY = [&]() { return GTABP ? GY(7) : fly; };
  auto FHY = [&]() { return GTABP ? GY(8) : fhy; };
  auto HCM0 = [&]() { return GTABP ? GX(9) : hcm0; };
  auto HCP0 = [&]() { return GTABP ? GX(10) : hcp0; };
  auto HCM1 = [&]() { return GTABP ? GX(11) * GY(0) : hcm1; };
  auto HCP1 = [&]() { return GTABP ? GX(11) * GY(1) : hcp1; };
  auto C2M = [&]() { return GTABP ? GX(11) * GY(4) : c2m; };
  auto HGR = [&]() { return GTABP ? GX(12) : hgr; };
  auto HAR = [&]() { return GTABP ? GX(13) : hAr; };
  auto HCGT = [&]() { return GTABP ? GX(11) * GY(9) : hcgt; };
  auto HCAT = [&]() { return GTABP ? GX(11) * GY(10) : hcAt; };
  auto HGX = [&]() { return GTABP ? GX(14) : hgx; };
  auto HGY = [&]() { return GTABP ? GY(11) : hgy; };
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int b = 0; b < 3; ++b) {
      mbar_expect_tx(&mbar[b], (uint32_t)SM::plane_bytes);
      tma_load_plane(&tmap, planes + b * PSTR, &mbar[b], xs, ys, k0 - 2 + b + NG);
    }
  }

  // raw conserved -> primitive of the cell at offset `off` of plane `pl`, in place if `store`
  // (gas + radiation EOS: Tg > 0 = a nearby temperature to start the solve from -- warp-collective, so only where all 32
  // lanes arrive together; Tout = the temperature found)
  auto convert = [&](double* pl, int off, double* Wout, bool store, bool coll = false, double Tg = 0.0, double* Tout = nullptr) {
    double U[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) U[v] = pl[v * FSTR + off];
    prim_of_cons<NV, EOS>(P, U, Wout, coll, Tg, Tout);
    if (store) {
#pragma unroll
      for (int v = 0; v < NV; ++v) pl[v * FSTR + off] = Wout[v];
    }
  };
  // own cell + the ghost cells this thread is responsible for (every needed cell of the box exactly once)
  auto convert_plane = [&](double* pl, double* Wown, bool coll = false, double Tg = 0.0, double* Tout = nullptr) {
    convert(pl, cidx, Wown, act, coll, Tg, Tout);
    if (xoff != 0 && act) {
      double tmp[NV];
      convert(pl, cidx + xoff, tmp, true, false, Tg);   // lane-divergent: the per-lane Newton loop, started from the neighbour's T
      if (coff != 0) convert(pl, cidx + coff, tmp, true, false, Tg);
    }
  };

  double dzm[NV];             // W(p) - W(p-1) of this column
  double Tcar = 0.0, Tprev = 0.0, Tul = 0.0;   // gas + radiation EOS: T^n of the own cell of plane p, of plane p-1, of the cell in Ul
  {
    double Wm2[NV], Wc0[NV];
    mbar_wait(&mbar[0], 0u);
    convert(planes, cidx, Wm2, false);
    mbar_wait(&mbar[1], 0u);
    phase = 3u;
    convert_plane(planes + PSTR, Wc0, false, 0.0, &Tcar);
#pragma unroll
    for (int v = 0; v < NV; ++v) dzm[v] = Wc0[v] - Wm2[v];
    __syncthreads();          // everyone has read plane k0-2: its buffer takes plane k0+1
    if (threadIdx.x == 0) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(&mbar[0], (uint32_t)SM::plane_bytes);
      tma_load_plane(&tmap, planes, &mbar[0], xs, ys, k0 + 1 + NG);
    }
  }

  double zp[NF];              // predicted state on the upper z face of the previous plane
  double Up[NV];              // partially updated cell of the previous plane
  double Un0 = 0.0, Unm[3] = {0.0, 0.0, 0.0};   // rho^n, m^n of the previous plane (time-centred gravity)
  double Ul[5] = {1.0, 0.0, 0.0, 0.0, 1.0};     // rho, m, E of the cell written one iteration ago (deferred CFL rate)
  bool st_l = false;                            // ... and whether it was stored
  double EA = 0.0, DV = 0.0, en_p = 1.0, Pn_p = 1.0;   // EMON: dt x (-div(u e)) and dt x div u of the previous plane's cell so far; its e^n, P^n
  double rate_max = 0.0;
  bool bad = false;
#pragma unroll
  for (int v = 0; v < NF; ++v) zp[v] = 1.0;
#pragma unroll
  for (int v = 0; v < NV; ++v) Up[v] = 1.0;
  double* outp = s.Uout + L.off(min(i, L.n[0] - 1) + NG, min(j, L.n[1] - 1) + NG, k0 - 2 + NG);   // cell (i, j, p-1) at p = k0-1

  // A7: CFL rate + positivity check of the cell in Ul (padded z index pkc).  e <= 0, or rho and e of opposite
  // sign, make the sound speed (hence the rate) NaN; both negative is caught by rho > 0.  It runs one iteration
  // after the cell was written so that its serial chain (1/rho -> e -> sqrt) overlaps the slope arithmetic.
  auto cfl_rate = [&](int pkc) {
    const double mm = fma(Ul[3], Ul[3], fma(Ul[2], Ul[2], Ul[1] * Ul[1]));
    const double ir = rcp3(Ul[0]);
    const double e = fma(-0.5 * ir, mm, Ul[4]);
    double cs;
    if (EOS == HX_EOS_IDEAL) {
      cs = sqrt3((P.gamma * P.gm1) * ir * e);
    } else {
      double pn;
      gr_from_energy_n<1>(P, &Ul[0], &ir, &e, &pn, &cs, Tul);   // warp-collective; e <= 0 gives T = NaN, hence a NaN sound speed, like the ideal branch
    }
    const double l0 = GTAB ? GX(5) : il0, l1 = GTAB ? GX(6) * GY(5) : il1, l2xy = GTAB ? GX(6) * GY(6) : il2xy;
    const double il2 = UNI ? a.uil[2] : l2xy * ZT(5, max(pkc, zb));
    const double rate = fma(fma(fabs(Ul[1]), ir, cs), l0, fma(fma(fabs(Ul[2]), ir, cs), l1, fma(fabs(Ul[3]), ir, cs) * il2));
    const bool fine = (Ul[0] > 0.0) && (rate < __longlong_as_double(0x7ff0000000000000LL));
    rate_max = (st_l && fine && rate > rate_max) ? rate : rate_max;
    bad = bad || (st_l && !fine);
  };

  // [B] O2-O4 for the cell of plane p: limited slopes, face states, half-step increment dU (Eq. 17-18, unsplit)
  // nvp_tag: how many leading fields it handles (all of them for the ring warps; the five hydro fields for the
  // owners, whose passive scalars follow one at a time to keep the register peak down); unc6: per-face signed
  // (dt/2) dS/dV u_n for that scalar pass.
  auto predictor = [&](auto nvp_tag, const double* Pc, const double* Wn, int pk, double* Wc, double* dU, double* Uxm, double* Uxp,
                       double* Uym, double* Uyp, double* Uzm, double* Uzp, double& hcm2, double* unc6, double& Tc, double& ec) {
    constexpr int NVP = decltype(nvp_tag)::value;
    double flz, fhz, hcp2;   // per-plane z geometry (uniform addresses)
    if (UNI) {
      flz = fhz = a.uf[2];
      hcm2 = hcp2 = a.uhc[2];
    } else {
      const double hwz = ZT(0, pk);
      flz = hwz * ZT(1, pk);
      fhz = hwz * ZT(1, pk + 1);
      hcm2 = C2M() * ZT(2, pk);
      hcp2 = (SPH ? C2M() : c2p) * ZT(3, pk);   // spherical: both z faces share the (r, theta) factors
    }
#pragma unroll
    for (int v = 0; v < NVP; ++v) {
      Wc[v] = Pc[v * FSTR + cidx];
      dU[v] = 0.0;
    }
    // gas + radiation EOS: temperature and internal energy of the cell centre, the Newton start of its twelve face solves
    Tc = 0.0;
    ec = 0.0;
    if (EOS != HX_EOS_IDEAL) {   // T of the cell centre was found when its plane was converted; e from Eq. 6a
      Tc = Tcar;
      ec = gr_energy_of_T(P, Wc[0], Tc);
    }
    double t[NVP];
    double uncl[6], pfl[6];     // gas + radiation EOS: per face (dt/2) dS/dV u_n and the face pressure
    double* const ul = unc6 ? unc6 : uncl;
    constexpr bool GR = EOS != HX_EOS_IDEAL;
    double dm[NVP], dp[NVP];    // one-sided differences of a direction (runtime-switch builds: all slopes of a direction behind one branch)
    if constexpr (LIM >= 0) {
#pragma unroll
      for (int v = 0; v < NVP; ++v) {
        const double wm = Pc[v * FSTR + cidx - 1], wp = Pc[v * FSTR + cidx + 1];
        t[v] = lim_pre<LIM, UNI>(P.limiter, Wc[v] - wm, wp - Wc[v], FLX(), FHX());
      }
    } else {
#pragma unroll
      for (int v = 0; v < NVP; ++v) {
        const double wm = Pc[v * FSTR + cidx - 1], wp = Pc[v * FSTR + cidx + 1];
        dm[v] = Wc[v] - wm;
        dp[v] = wp - Wc[v];
      }
      const double fl = FLX(), fh = FHX();
      lim_pre_n<NVP, LIM, UNI>(P.limiter, dm, dp, &fl, &fh, t);
    }
    face_cons_flux<NVP, 0, EOS>(P, Wc, t, UNI ? -FLX() : -lim_scale<LIM>(), HCM0(), Uxm, dU, (unc6 || GR) ? ul + 0 : nullptr, pfl + 0);
    face_cons_flux<NVP, 0, EOS>(P, Wc, t, UNI ? FLX() : lim_scale<LIM>(), -HCP0(), Uxp, dU, (unc6 || GR) ? ul + 1 : nullptr, pfl + 1);
    if constexpr (LIM >= 0) {
#pragma unroll
      for (int v = 0; v < NVP; ++v) {
        const double wm = Pc[v * FSTR + cidx - PX], wp = Pc[v * FSTR + cidx + PX];
        t[v] = lim_pre<LIM, UNI>(P.limiter, Wc[v] - wm, wp - Wc[v], FLY(), FHY());
      }
    } else {
#pragma unroll
      for (int v = 0; v < NVP; ++v) {
        const double wm = Pc[v * FSTR + cidx - PX], wp = Pc[v * FSTR + cidx + PX];
        dm[v] = Wc[v] - wm;
        dp[v] = wp - Wc[v];
      }
      const double fl = FLY(), fh = FHY();
      lim_pre_n<NVP, LIM, UNI>(P.limiter, dm, dp, &fl, &fh, t);
    }
    face_cons_flux<NVP, 1, EOS>(P, Wc, t, UNI ? -FLY() : -lim_scale<LIM>(), HCM1(), Uym, dU, (unc6 || GR) ? ul + 2 : nullptr, pfl + 2);
    face_cons_flux<NVP, 1, EOS>(P, Wc, t, UNI ? FLY() : lim_scale<LIM>(), -HCP1(), Uyp, dU, (unc6 || GR) ? ul + 3 : nullptr, pfl + 3);
    if constexpr (LIM >= 0) {
#pragma unroll
      for (int v = 0; v < NVP; ++v) {
        const double dpz = Wn[v] - Wc[v];
        t[v] = lim_pre<LIM, UNI>(P.limiter, dzm[v], dpz, flz, fhz);
        dzm[v] = dpz;
      }
    } else {
#pragma unroll
      for (int v = 0; v < NVP; ++v) dp[v] = Wn[v] - Wc[v];
      lim_pre_n<NVP, LIM, UNI>(P.limiter, dzm, dp, &flz, &fhz, t);
#pragma unroll
      for (int v = 0; v < NVP; ++v) dzm[v] = dp[v];
    }
    face_cons_flux<NVP, 2, EOS>(P, Wc, t, UNI ? -flz : -lim_scale<LIM>(), hcm2, Uzm, dU, (unc6 || GR) ? ul + 4 : nullptr, pfl + 4);
    face_cons_flux<NVP, 2, EOS>(P, Wc, t, UNI ? flz : lim_scale<LIM>(), -hcp2, Uzp, dU, (unc6 || GR) ? ul + 5 : nullptr, pfl + 5);
    if (GR) {   // internal energies of the six face states (P -> T -> e, Eq. 6), all at once, into E and the energy flux
      const double rf[6] = {Uxm[0], Uxp[0], Uym[0], Uyp[0], Uzm[0], Uzp[0]};
      double ef[6];
      gr_energy_n<6>(P, rf, pfl, Tc, ef);
      Uxm[4] += ef[0];
      Uxp[4] += ef[1];
      Uym[4] += ef[2];
      Uyp[4] += ef[3];
      Uzm[4] += ef[4];
      Uzp[4] += ef[5];
#pragma unroll
      for (int k = 0; k < 6; ++k) dU[4] = fma(ef[k], ul[k], dU[4]);
    }
    const double rho = Wc[0];
    const double mcx = rho * Wc[1], mcy = rho * Wc[2], mcz = rho * Wc[3];
    if (SPH) {   // cell-centred geometric sources (R8)
      const double ur = Wc[1], ut = Wc[2], up = Wc[3], pr = Wc[4];
      dU[1] = fma(fma(mcy, ut, fma(mcz, up, 2.0 * pr)), HGR(), dU[1]);
      dU[2] += fma(mcz, up, pr) * HCGT() - mcy * ur * HAR();
      dU[3] -= mcz * fma(ur, HAR(), ut * HCAT());
    }
    if (grav_has(GRAV, 0)) {
      dU[1] = fma(rho, HGX(), dU[1]);
      dU[4] = fma(mcx, HGX(), dU[4]);
    }
    if (grav_has(GRAV, 1)) {
      dU[2] = fma(rho, HGY(), dU[2]);
      dU[4] = fma(mcy, HGY(), dU[4]);
    }
    if (grav_has(GRAV, 2, SPH)) {
      const double hgz = hdt * ZT(4, pk);
      dU[3] = fma(rho, hgz, dU[3]);
      dU[4] = fma(mcz, hgz, dU[4]);
    }
    if (lim_none) {
#pragma unroll
      for (int v = 0; v < NVP; ++v) dU[v] = 0.0;
    }
  };

  constexpr bool HLLC_STATIC = (RS == HX_RIEMANN_HLLC);
  auto march = [&](auto own_tag) {
  constexpr bool OWN = decltype(own_tag)::value;
  int bc = 1;                 // buffer of plane p
  int xyo = 0;                // ONEBAR: offset of this plane's exchange buffer (toggles between the two parity buffers)
  constexpr int UNR = HX_T2_UNROLL;
#pragma unroll UNR
  for (int p = k0 - 1; p <= k1; ++p, outp += L.sz) {
    const int pk = p + NG;
    const int bn = (bc == 2) ? 0 : bc + 1;
    double* Pc = planes + bc * PSTR;
    double* Pn = planes + bn * PSTR;
    double* const X = XY0 + xyo;                          // exchange slots of this plane
    double* const Y = X + NF * XSTR;
    double* const Xo = XY0 + (ONEBAR ? SM::XYSTR - xyo : 0);   // ... and of the previous plane (fluxes through its upper x / y faces)
    double* const Yo = Xo + NF * XSTR;
    if (ONEBAR) xyo = SM::XYSTR - xyo;
    mbar_wait(&mbar[bn], (phase >> bn) & 1u);            // plane p+1 has arrived (issued a whole iteration ago)
    phase ^= (1u << bn);

    // Edge iterations (p = k0-1 and p = k1) run the same code on valid but unused data; only the global
    // store and the CFL rate are predicated, so the iteration is three straight-line blocks.
    double Wn[NV], Wc[NV], dU[NV], hcm2, Tc, ec, Tn = 0.0;
    double Uf[6][NV];          // conserved face states: 0 x-, 1 x+, 2 y-, 3 y+, 4 z-, 5 z+
    if constexpr (OWN) {
      // ======== block 1: slopes, half-step increment, the six predicted states in two interleaved
      // batches, the deferred CFL rate of cell p-2 =============================================================
      cfl_rate(pk - 2);
      convert(Pn, cidx, Wn, true, true, Tcar, &Tn);            // [A] cons -> prim of the own cell of plane p+1, in place (T started from the cell below)
      double unc[6], ir6[6];   // per face: signed (dt/2) dS/dV u_n of the face state, 1/rho of the predicted state
      predictor(std::integral_constant<int, 5>{}, Pc, Wn, pk, Wc, dU, Uf[0], Uf[1], Uf[2], Uf[3], Uf[4], Uf[5], hcm2, unc, Tc, ec);
      double qxm[NF], qym[NF], qzm[NF], zpn[NF];
      {
        double qa[NF], qb[NF];
        const double* const ua[3] = {Uf[1], Uf[3], Uf[4]};
        double* const qo[3] = {qa, qb, qzm};
        double* const io[3] = {&ir6[1], &ir6[3], &ir6[4]};
        pred_states<5, 3, EOS>(P, ua, dU, qo, io, Tc);
#pragma unroll
        for (int v = 0; v < 7; ++v) {
          X[v * XSTR + xs_own] = qa[v];
          Y[v * YSTR + ys_own] = qb[v];
        }
      }
      {
        const double* const ub[3] = {Uf[0], Uf[2], Uf[5]};
        double* const qo[3] = {qxm, qym, zpn};
        double* const io[3] = {&ir6[0], &ir6[2], &ir6[5]};
        pred_states<5, 3, EOS>(P, ub, dU, qo, io, Tc);
      }
      double Un[NV];           // U^n of cell p
      {
        const double rho = Wc[0];
        Un[0] = rho;
        Un[1] = rho * Wc[1];
        Un[2] = rho * Wc[2];
        Un[3] = rho * Wc[3];
        Un[4] = fma(0.5, fma(Un[3], Wc[3], fma(Un[2], Wc[2], Un[1] * Wc[1])), EOS == HX_EOS_IDEAL ? Wc[4] * P.igm1 : ec);
      }
      const double Pn_c = Wc[4], en_c = (EOS == HX_EOS_IDEAL) ? Wc[4] * P.igm1 : ec;   // EMON: P^n, e^n of cell p
      if constexpr (NV > 5) {
        // Passive scalars one at a time (R7: mass fractions are reconstructed, rho f is advanced): limited slopes,
        // the six face values, the scalar's own half-step increment from the face mass fluxes kept in `unc`, and
        // the predicted mass fraction on every face.  Same arithmetic as the all-fields predictor of the ring path.
        double flz, fhz;
        if (UNI) {
          flz = fhz = a.uf[2];
        } else {
          const double hwz = ZT(0, pk);
          flz = hwz * ZT(1, pk);
          fhz = hwz * ZT(1, pk + 1);
        }
        const double scx = UNI ? FLX() : lim_scale<LIM>(), scy = UNI ? FLY() : lim_scale<LIM>(), scz = UNI ? flz : lim_scale<LIM>();
#pragma unroll
        for (int sv = 5; sv < NV; ++sv) {
          const double* Ps = Pc + sv * FSTR + cidx;
          const double fc = Ps[0];
          const double dp = Pn[sv * FSTR + cidx] - fc;
          double tx, ty, tz;
          if constexpr (LIM >= 0) {
            tx = lim_pre<LIM, UNI>(P.limiter, fc - Ps[-1], Ps[1] - fc, FLX(), FHX());
            ty = lim_pre<LIM, UNI>(P.limiter, fc - Ps[-PX], Ps[PX] - fc, FLY(), FHY());
            tz = lim_pre<LIM, UNI>(P.limiter, dzm[sv], dp, flz, fhz);
          } else {
            const double dm3[3] = {fc - Ps[-1], fc - Ps[-PX], dzm[sv]}, dp3[3] = {Ps[1] - fc, Ps[PX] - fc, dp};
            const double fl3[3] = {FLX(), FLY(), flz}, fh3[3] = {FHX(), FHY(), fhz};
            double t3[3];
            lim_pre_n<3, LIM, UNI, true>(P.limiter, dm3, dp3, fl3, fh3, t3);
            tx = t3[0], ty = t3[1], tz = t3[2];
          }
          dzm[sv] = dp;
          double rf[6];
          rf[0] = Uf[0][0] * fma(-scx, tx, fc);
          rf[1] = Uf[1][0] * fma(scx, tx, fc);
          rf[2] = Uf[2][0] * fma(-scy, ty, fc);
          rf[3] = Uf[3][0] * fma(scy, ty, fc);
          rf[4] = Uf[4][0] * fma(-scz, tz, fc);
          rf[5] = Uf[5][0] * fma(scz, tz, fc);
          double dUs = 0.0;
#pragma unroll
          for (int k = 0; k < 6; ++k) dUs = fma(rf[k], unc[k], dUs);
          if (lim_none) dUs = 0.0;
          X[(2 + sv) * XSTR + xs_own] = (rf[1] + dUs) * ir6[1];
          Y[(2 + sv) * YSTR + ys_own] = (rf[3] + dUs) * ir6[3];
          if (SM::NPRIV > 0) {
            constexpr int PS = TY * TX;
            priv[(4 * (sv - 5) + 0) * PS] = (rf[0] + dUs) * ir6[0];
            priv[(4 * (sv - 5) + 1) * PS] = (rf[2] + dUs) * ir6[2];
            priv[(4 * (sv - 5) + 2) * PS] = (rf[4] + dUs) * ir6[4];
            priv[(4 * (sv - 5) + 3) * PS] = (rf[5] + dUs) * ir6[5];
          } else {
            qxm[2 + sv] = (rf[0] + dUs) * ir6[0];
            qym[2 + sv] = (rf[2] + dUs) * ir6[2];
            qzm[2 + sv] = (rf[4] + dUs) * ir6[4];
            zpn[2 + sv] = (rf[5] + dUs) * ir6[5];
          }
          Un[sv] = Wc[0] * fc;
        }
      }
      asm volatile("bar.sync 0;" ::: "memory");          // (1) "+" states visible; all reads of plane p done
      if (threadIdx.x == 0 && p + 3 <= k1 + 1) {         // plane p+3 takes the buffer of plane p
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(&mbar[bc], (uint32_t)SM::plane_bytes);
        tma_load_plane(&tmap, Pc, &mbar[bc], xs, ys, p + 3 + NG);
      }
      // ======== block 2: the three Riemann problems on the lower faces of this cell (x and y fluxes go back into
      // the slots), finish cell p-1 with the z flux, start cell p =============================================
      if (SM::NPRIV > 0) {
        constexpr int PS = TY * TX;
#pragma unroll
        for (int sv = 5; sv < NV; ++sv) {
          qxm[2 + sv] = priv[(4 * (sv - 5) + 0) * PS];
          qym[2 + sv] = priv[(4 * (sv - 5) + 1) * PS];
          qzm[2 + sv] = priv[(4 * (sv - 5) + 2) * PS];
          zpn[2 + sv] = priv[(4 * (sv - 5) + 3) * PS];
        }
      }
      // fluxes through the upper x and y faces of a cell come back in its own slots (written by the neighbours across
      // those faces): into the partially updated cell Up
      auto upper_xy = [&](const double* Xs, const double* Ys) {
        struct { double p0, xp, p1, yp; } Kp;
        Kp.p0 = GTAB ? GX(1) : k0p;
        Kp.xp = GTAB ? GX(3) : kxp;
        Kp.p1 = GTAB ? GX(4) * GY(1) : k1p;
        Kp.yp = GTAB ? GX(4) * GY(3) : kyp;
        if (EMON) {
          EA -= fma(Kp.p0, Xs[NV * XSTR + xs_own], Kp.p1 * Ys[NV * YSTR + ys_own]);
          DV += fma(Kp.p0, Xs[(NV + 1) * XSTR + xs_own], Kp.p1 * Ys[(NV + 1) * YSTR + ys_own]);
        }
#pragma unroll
        for (int v = 0; v < NV; ++v) Up[v] = fma(-((SPH && (v == 2 || v == 3)) ? Kp.xp : Kp.p0), Xs[v * XSTR + xs_own], Up[v]);
        if (SPH) Up[1] = fma(HGR(), Ys[2 * YSTR + ys_own], Up[1]);
#pragma unroll
        for (int v = 0; v < NV; ++v) Up[v] = fma(-((SPH && v == 3) ? Kp.yp : Kp.p1), Ys[v * YSTR + ys_own], Up[v]);
      };
      if (ONEBAR) upper_xy(Xo, Yo);                      // cell p-1: its neighbours wrote these during the previous plane, before barrier (1)
      double Fx[NV], Fy[NV], Fz[NV];
      double phx = 0.0, ufx = 0.0, phy = 0.0, ufy = 0.0, phz = 0.0, ufz = 0.0;
      {
        double qlx[NF], qly[NF];
#pragma unroll
        for (int v = 0; v < NF; ++v) {
          qlx[v] = X[v * XSTR + xs_nbr];
          qly[v] = Y[v * YSTR + ys_nbr];
        }
        if (HLLC_STATIC || (RS < 0 && P.riemann == HX_RIEMANN_HLLC)) {
          const int dirs[3] = {0, 1, 2};
          const double* const Ls[3] = {qlx, qly, zp};
          const double* const Rs[3] = {qxm, qym, qzm};
          double* const Fs[3] = {Fx, Fy, Fz};
          hllc_n<NV, 3>(dirs, Ls, Rs, Fs);
        } else {
          riemann_fs<NV, RS, 0>(P, qlx, qxm, Fx);
          riemann_fs<NV, RS, 1>(P, qly, qym, Fy);
          riemann_fs<NV, RS, 2>(P, zp, qzm, Fz);
        }
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          X[v * XSTR + xs_nbr] = Fx[v];
          Y[v * YSTR + ys_nbr] = Fy[v];
        }
        if (EMON) {   // Eq. 10: advective flux of e and face velocity of the three lower faces; x and y ones ride in the two spare slot fields
          monitor_rec<0>(qlx, qxm, Fx[0], phx, ufx);
          monitor_rec<1>(qly, qym, Fy[0], phy, ufy);
          monitor_rec<2>(zp, qzm, Fz[0], phz, ufz);
          X[NV * XSTR + xs_nbr] = phx;
          X[(NV + 1) * XSTR + xs_nbr] = ufx;
          Y[NV * YSTR + ys_nbr] = phy;
          Y[(NV + 1) * YSTR + ys_nbr] = ufy;
        }
      }
#pragma unroll
      for (int v = 0; v < NF; ++v) zp[v] = zpn[v];
      {   // the flux through the upper z face of cell p-1 is Fz: write the cell once
        const double k2p = UNI ? 2.0 * a.uhc[2] : (GTAB ? GX(4) * GY(4) * ZT(3, pk - 1) : 2.0 * c2p * ZT(3, pk - 1));
        double Unew[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) Unew[v] = fma(-k2p, Fz[v], Up[v]);
        if (SPH) {   // upper phi-face half of F^phi_phi in S_r and S_theta (Eq. 16 as read in R10, R11)
          Unew[1] = fma(HGR(), Fz[3], Unew[1]);
          Unew[2] = fma(HCGT(), Fz[3], Unew[2]);
        }
        if (GRAV != GRAV_OFF) {   // time-centred (R13)
          const double rs = Un0 + Unew[0];
          if (grav_has(GRAV, 0)) {
            const double m1 = fma(rs, HGX(), Unew[1]);
            Unew[4] = fma(Unm[0] + m1, HGX(), Unew[4]);
            Unew[1] = m1;
          }
          if (grav_has(GRAV, 1)) {
            const double m2 = fma(rs, HGY(), Unew[2]);
            Unew[4] = fma(Unm[1] + m2, HGY(), Unew[4]);
            Unew[2] = m2;
          }
          if (grav_has(GRAV, 2, SPH)) {
            const double hgzp = hdt * ZT(4, pk - 1);
            const double m3 = fma(rs, hgzp, Unew[3]);
            Unew[4] = fma(Unm[2] + m3, hgzp, Unew[4]);
            Unew[3] = m3;
          }
        }
        if (EMON) {   // Eq. 11-12 for cell p-1: e1 from the total energy, e2 from Eq. 10 (dt folded into the coefficients), E reset
          const double eaf = fma(-k2p, phz, EA), dvf = fma(k2p, ufz, DV);
          const double ek = 0.5 * fma(Unew[3], Unew[3], fma(Unew[2], Unew[2], Unew[1] * Unew[1])) * rcp3(Unew[0]);
          const double e1 = Unew[4] - ek, e2 = en_p + fma(-Pn_p, dvf, eaf);
          Unew[4] = ek + monitor_blend2(P.emon_eps, en_p, e1, e2, ek);
        }
        st_l = st_ok && (p > k0);
        if (st_l) {
#pragma unroll
          for (int v = 0; v < NV; ++v) outp[v * L.sv] = Unew[v];
          if (XG && xedge) {   // x-ghost images of this cell (R16: both null-gradient layers copy the boundary cell; reflecting: mirror, -m_x)
            const int n0 = L.n[0];
            auto put = [&](int off, bool neg) {
#pragma unroll
              for (int v = 0; v < NV; ++v) outp[v * L.sv + off] = (v == 1 && neg) ? -Unew[v] : Unew[v];
            };
            if (i < NG) {                                  // one of the first two cells
              if (a.bcx_hi == HX_BC_PERIODIC) put(n0, false);
              if (a.bcx_lo == HX_BC_TRANSMISSIVE) {
                if (i == 0) {
                  put(-1, false);
                  put(-2, false);
                }
              } else if (a.bcx_lo != HX_BC_PERIODIC) put(-1 - 2 * i, true);
            }
            if (i >= n0 - NG) {                            // one of the last two cells
              if (a.bcx_lo == HX_BC_PERIODIC) put(-n0, false);
              if (a.bcx_hi == HX_BC_TRANSMISSIVE) {
                if (i == n0 - 1) {
                  put(1, false);
                  put(2, false);
                }
              } else if (a.bcx_hi != HX_BC_PERIODIC) put(2 * (n0 - 1 - i) + 1, true);
            }
          }
        }
#pragma unroll
        for (int v = 0; v < 5; ++v) Ul[v] = Unew[v];
        if (EOS != HX_EOS_IDEAL) Tul = Tprev;              // T^n of cell p-1: where the solve for its new temperature starts
      }
      {   // cell p: U^n + the three lower faces
        const double k2m = 2.0 * hcm2;
        struct { double m0, xm, m1, ym; } K;   // dt dS/dV of the lower x and y faces (spherical: from the column / row tables)
        K.m0 = GTAB ? GX(0) : k0m;
        K.xm = GTAB ? GX(2) : kxm;
        K.m1 = GTAB ? GX(4) * GY(0) : k1m;
        K.ym = GTAB ? GX(4) * GY(2) : kym;
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          double u = fma(k2m, Fz[v], Un[v]);
          u = fma((SPH && (v == 2 || v == 3)) ? K.xm : K.m0, Fx[v], u);
          Up[v] = fma((SPH && v == 3) ? K.ym : K.m1, Fy[v], u);
        }
        if (SPH) {
          Up[1] = fma(HGR(), Fz[3] + Fy[2], Up[1]);
          Up[2] = fma(HCGT(), Fz[3], Up[2]);
        }
        if (GRAV != GRAV_OFF) {
          Un0 = Un[0];
          if (grav_has(GRAV, 0)) Unm[0] = Un[1];
          if (grav_has(GRAV, 1)) Unm[1] = Un[2];
          if (grav_has(GRAV, 2, SPH)) Unm[2] = Un[3];
        }
        if (EMON) {
          EA = fma(k2m, phz, fma(K.m0, phx, K.m1 * phy));
          DV = -fma(k2m, ufz, fma(K.m0, ufx, K.m1 * ufy));
          en_p = en_c;
          Pn_p = Pn_c;
        }
      }
      if (!ONEBAR) {
        asm volatile("bar.sync 0;" ::: "memory");        // (2) fluxes visible
        upper_xy(X, Y);                                  // block 3: fluxes through the upper x and y faces of cell p
      }
    } else {
      // ======== ring warps: predictor, one predicted state, at most one Riemann solve =====================
      convert_plane(Pn, Wn, true, Tcar, &Tn);
      double q[NF];
      if constexpr (RING2) {
        // many fields: like the owners, the five hydro fields first and then the passive scalars one at a time (same
        // arithmetic as the owner path), so that the ring path stays within its small register budget
        double unc[6], irs;
        predictor(std::integral_constant<int, 5>{}, Pc, Wn, pk, Wc, dU, Uf[0], Uf[1], Uf[2], Uf[3], Uf[4], Uf[5], hcm2, unc, Tc, ec);
        const int ks = (wid == TY) ? 3 : ((wid == TY + 1) ? 2 : ((wid == TY + 2) ? 1 : 0));   // the face whose predicted state this warp provides
        {
          double Usel[5];
#pragma unroll
          for (int v = 0; v < 5; ++v) Usel[v] = (ks & 2) ? ((ks & 1) ? Uf[3][v] : Uf[2][v]) : ((ks & 1) ? Uf[1][v] : Uf[0][v]);
          const double* const us[1] = {Usel};
          double* const qo[1] = {q};
          double* const io[1] = {&irs};
          pred_states<5, 1, EOS>(P, us, dU, qo, io, Tc);
        }
        double flz, fhz;
        if (UNI) {
          flz = fhz = a.uf[2];
        } else {
          const double hwz = ZT(0, pk);
          flz = hwz * ZT(1, pk);
          fhz = hwz * ZT(1, pk + 1);
        }
        const double scx = UNI ? FLX() : lim_scale<LIM>(), scy = UNI ? FLY() : lim_scale<LIM>(), scz = UNI ? flz : lim_scale<LIM>();
#pragma unroll
        for (int sv = 5; sv < NV; ++sv) {
          const double* Ps = Pc + sv * FSTR + cidx;
          const double fc = Ps[0];
          const double dp = Pn[sv * FSTR + cidx] - fc;
          double tx, ty, tz;
          if constexpr (LIM >= 0) {
            tx = lim_pre<LIM, UNI>(P.limiter, fc - Ps[-1], Ps[1] - fc, FLX(), FHX());
            ty = lim_pre<LIM, UNI>(P.limiter, fc - Ps[-PX], Ps[PX] - fc, FLY(), FHY());
            tz = lim_pre<LIM, UNI>(P.limiter, dzm[sv], dp, flz, fhz);
          } else {
            const double dm3[3] = {fc - Ps[-1], fc - Ps[-PX], dzm[sv]}, dp3[3] = {Ps[1] - fc, Ps[PX] - fc, dp};
            const double fl3[3] = {FLX(), FLY(), flz}, fh3[3] = {FHX(), FHY(), fhz};
            double t3[3];
            lim_pre_n<3, LIM, UNI, true>(P.limiter, dm3, dp3, fl3, fh3, t3);
            tx = t3[0], ty = t3[1], tz = t3[2];
          }
          dzm[sv] = dp;
          double rf[6];
          rf[0] = Uf[0][0] * fma(-scx, tx, fc);
          rf[1] = Uf[1][0] * fma(scx, tx, fc);
          rf[2] = Uf[2][0] * fma(-scy, ty, fc);
          rf[3] = Uf[3][0] * fma(scy, ty, fc);
          rf[4] = Uf[4][0] * fma(-scz, tz, fc);
          rf[5] = Uf[5][0] * fma(scz, tz, fc);
          double dUs = 0.0;
#pragma unroll
          for (int k = 0; k < 6; ++k) dUs = fma(rf[k], unc[k], dUs);
          if (lim_none) dUs = 0.0;
          const double rsel = (ks & 2) ? ((ks & 1) ? rf[3] : rf[2]) : ((ks & 1) ? rf[1] : rf[0]);
          q[2 + sv] = (rsel + dUs) * irs;
        }
        if (wid == TY) {
#pragma unroll
          for (int v = 0; v < NF; ++v) Y[v * YSTR + ys_own] = q[v];
        } else if (wid == TY + 2 && act) {
#pragma unroll
          for (int v = 0; v < NF; ++v) X[v * XSTR + xs_own] = q[v];
        }
      } else {
      predictor(std::integral_constant<int, NV>{}, Pc, Wn, pk, Wc, dU, Uf[0], Uf[1], Uf[2], Uf[3], Uf[4], Uf[5], hcm2, nullptr, Tc, ec);
      if (wid == TY) {
        pred_state<NV, EOS>(P, Uf[3], dU, q, Tc);
#pragma unroll
        for (int v = 0; v < NF; ++v) Y[v * YSTR + ys_own] = q[v];
      } else if (wid == TY + 1) {
        pred_state<NV, EOS>(P, Uf[2], dU, q, Tc);
      } else if (wid == TY + 2) {
        pred_state<NV, EOS>(P, Uf[1], dU, q, Tc);
        if (act) {
#pragma unroll
          for (int v = 0; v < NF; ++v) X[v * XSTR + xs_own] = q[v];
        }
      } else {
        pred_state<NV, EOS>(P, Uf[0], dU, q, Tc);
      }
      }
      asm volatile("bar.sync 0;" ::: "memory");          // (1)
      if (wid == TY + 1) {
        double ql[NF], F[NV];
#pragma unroll
        for (int v = 0; v < NF; ++v) ql[v] = Y[v * YSTR + ys_nbr];
        riemann_fs<NV, RS, 1>(P, ql, q, F);
#pragma unroll
        for (int v = 0; v < NV; ++v) Y[v * YSTR + ys_nbr] = F[v];
        if (EMON) {
          double ph, uf;
          monitor_rec<1>(ql, q, F[0], ph, uf);
          Y[NV * YSTR + ys_nbr] = ph;
          Y[(NV + 1) * YSTR + ys_nbr] = uf;
        }
      } else if (wid == TY + 3 && act) {
        double ql[NF], F[NV];
#pragma unroll
        for (int v = 0; v < NF; ++v) ql[v] = X[v * XSTR + xs_nbr];
        riemann_fs<NV, RS, 0>(P, ql, q, F);
#pragma unroll
        for (int v = 0; v < NV; ++v) X[v * XSTR + xs_nbr] = F[v];
        if (EMON) {
          double ph, uf;
          monitor_rec<0>(ql, q, F[0], ph, uf);
          X[NV * XSTR + xs_nbr] = ph;
          X[(NV + 1) * XSTR + xs_nbr] = uf;
        }
      }
      if (!ONEBAR) asm volatile("bar.sync 0;" ::: "memory");   // (2)
    }
    bc = bn;
    if (EOS != HX_EOS_IDEAL) {
      Tprev = Tcar;
      Tcar = Tn;
    }
  }
  };
  if (owner) {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(owner_regs(SPH, NV, TY)));
    march(std::true_type{});
    cfl_rate(k1 + 1 + NG - 2);                           // the last cell written (plane k1-1)
  } else {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(ring_regs(SPH, NV, TY)));
    march(std::false_type{});
  }

  if (bad) atomicOr(s.status, 1);
  block_rate_max(rate_max, s.rate_bits);
}

}  // namespace t2
}  // namespace hx

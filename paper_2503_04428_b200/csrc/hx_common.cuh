// hx_common.cuh -- shared declarations of the CUDA path (layout, geometry tables, pointwise physics).
// Hand-written for sm_100a.  Shares nothing with oracle/.
//
// Pointwise physics follows PAPER.md: Eq. 1 + Eq. 5 (cons <-> prim, ideal gas), Eq. 17 (limited
// slopes), Eq. 18 (Hancock predictor), Eq. 19 with HLL / HLLC (L197-L201), readings R1-R25 of DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#include "../../include/hx.h"

namespace hx {

constexpr int NG = 2;                 // ghost layers per face in active directions
constexpr int NVMAX = HX_MAX_NVAR;

// Padded structure-of-arrays layout [nvar][np2][np1][pitch0]; offsets in doubles.
struct Layout {
  int ndim, nvar;
  int n[3];    // interior cells
  int ng[3];   // NG for active directions, 0 otherwise
  int np[3];   // n + 2 ng
  int lead;    // doubles of padding in front of each x row (alignment of the first interior cell)
  long long sy, sz, sv;   // strides of j, k, variable
  __host__ __device__ long long off(int pi, int pj, int pk) const { return (long long)pk * sz + (long long)pj * sy + pi + lead; }
};

// 1-D geometry tables, all indexed by the padded cell index of their axis.
// Face-area / volume ratios are products of per-axis factors:
//   dS_{d,-}/dV = cf[d][0][0][pi] * cf[d][0][1][pj] * cf[d][0][2][pk],   dS_{d,+}/dV likewise with cf[d][1].
// CFL lengths: 1/l_d = lf[d][0][pi] * lf[d][1][pj] * lf[d][2][pk].
struct Tables {
  const double* cf[3][2][3];
  const double* lf[3][3];
  const double* idx[3];   // idx[d][p] = 1 / (xc[p] - xc[p-1])   (p >= 1)
  const double* hw[3];    // half cell width
  const double* grav[3];  // acceleration component along d seen by cell p (mirrored behind reflecting faces, R25)
  // spherical source factors
  const double* gr;   // by i: (dS^r+ - dS^r-)/(2 dV)
  const double* Ar;   // by i: (r+ - r-)(dS^r+ + dS^r-)/((r+ + r-) dV)
  const double* rr;   // by i: (r+ - r-)/(r+ + r-)
  const double* cr;   // by i: ((r+^2 - r-^2)/2) / ((r+^3 - r-^3)/3)
  const double* gt;   // by j: (sin th+ - sin th-)/(cos th- - cos th+)
  const double* At;   // by j: st * (sin th+ + sin th-)/(cos th- - cos th+)
  const double* st;   // by j: (sin th+ - sin th-)/(sin th+ + sin th-)
};

struct Phys {
  double gamma, gm1, igm1;
  int limiter, riemann, gravity, spherical;
  int eos;                // HX_EOS_IDEAL or HX_EOS_GAS_RADIATION
  double rgas, arad;      // gas + radiation: k_b / mu and the radiation constant a_r (Eq. 6a-6b)
  double emon_eps;        // > 0: internal-energy monitoring (Eq. 10-12) with this epsilon
};

struct StepArgs {
  Layout L;
  Tables T;
  Phys P;
  const double* __restrict__ Uin;
  double* __restrict__ Uout;
  double dt;
  unsigned long long* rate_bits;   // max over cells of the CFL rate of the NEW state (bit pattern of a double >= 0)
  int* status;                     // bit 0: non-physical state seen
};

// ---------------------------------------------------------------------------------------------
// Limiters (Eq. 17; R3-R5).  a = backward gradient, b = forward gradient.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double limited_slope(int lim, double a, double b) {
  if (lim == HX_LIM_NONE) return 0.0;
  const double ab = a * b;
  if (!(ab > 0.0)) return 0.0;
  const double fa = fabs(a), fb = fabs(b);
  double s;
  switch (lim) {
    case HX_LIM_MINMOD: s = fmin(fa, fb); break;
    case HX_LIM_VANLEER: s = 2.0 * fa * fb / (fa + fb); break;
    case HX_LIM_VANALBADA: s = fa * fb * (fa + fb) / (fa * fa + fb * fb); break;
    default: s = fmin(fmin(2.0 * fa, 2.0 * fb), 0.5 * (fa + fb)); break;   // MC
  }
  return copysign(s, a);
}

// ---------------------------------------------------------------------------------------------
// Equation of state.  Ideal gas: Eq. 5.  Ideal gas in equilibrium with radiation (Eq. 6-7):
//   e = rho (k_b/mu) T / (gamma-1) + a_r T^4,   P = rho (k_b/mu) T + a_r T^4 / 3,   alpha = P_r / P_g,
//   c_s^2 = (gamma/(gamma-1) + 20 alpha + 16 alpha^2) / (1/(gamma-1) + 12 alpha) * P_g / rho.
// T comes from e (or from P) by Newton-Raphson, as the paper prescribes; started at the smaller of the two
// single-term roots the iterate can only move down towards the root; it stops when the correction is a few ulp.
// ---------------------------------------------------------------------------------------------
static __device__ __noinline__ double temperature_root(double a1, double a4, double b) {   // not inlined: keeps the generic kernels small (compile time)   // a1 T + a4 T^4 = b
  // non-physical (e <= 0 or P <= 0): NaN, so that P, c_s and the CFL rate come out NaN and the callers' checks report it.
  // (A negative T = b / a1 would NOT do: P = a_r T^4 / 3 + rho R T is positive again once a_r |T|^3 > 3 rho R.)
  if (!(b > 0.0)) return __longlong_as_double(0x7ff8000000000000LL);
  double T = fmin(b / a1, sqrt(sqrt(b / a4)));
  for (int it = 0; it < 60; ++it) {                    // R27: until the correction is a few ulp; quadratic, ~5-9 steps
    const double T3 = T * T * T;
    const double step = (fma(a4 * T3, T, a1 * T) - b) / fma(4.0 * a4, T3, a1);
    T -= step;
    if (fabs(step) <= 1e-15 * T) break;
  }
  return T;
}

__device__ __forceinline__ double eos_pressure(const Phys& P, double rho, double e) {
  if (P.eos == HX_EOS_IDEAL) return P.gm1 * e;
  const double T = temperature_root(rho * P.rgas * P.igm1, P.arad, e);
  const double T2 = T * T;
  return fma(P.arad * (1.0 / 3.0), T2 * T2, rho * P.rgas * T);
}

__device__ __forceinline__ double eos_energy(const Phys& P, double rho, double p) {
  if (P.eos == HX_EOS_IDEAL) return p * P.igm1;
  const double T = temperature_root(rho * P.rgas, P.arad * (1.0 / 3.0), p);
  const double T2 = T * T;
  return fma(P.arad, T2 * T2, rho * P.rgas * T * P.igm1);
}

__device__ __forceinline__ double eos_sound_speed(const Phys& P, double rho, double p) {
  if (P.eos == HX_EOS_IDEAL) return sqrt(P.gamma * p / rho);
  const double T = temperature_root(rho * P.rgas, P.arad * (1.0 / 3.0), p);
  const double T2 = T * T;
  const double pg = rho * P.rgas * T, al = P.arad * (1.0 / 3.0) * T2 * T2 / pg;
  return sqrt((P.gamma * P.igm1 + al * (20.0 + 16.0 * al)) / (P.igm1 + 12.0 * al) * pg / rho);
}

// ---------------------------------------------------------------------------------------------
// cons <-> prim (Eq. 1, Eq. 5 / 6).  Field order: rho, m_d / u_d (ND of them), E / P, scalars.
// ---------------------------------------------------------------------------------------------
template <int ND>
__device__ __forceinline__ void cons_to_prim(const Phys& P, int nv, const double* U, double* W) {
  const double rho = U[0];
  const double ir = 1.0 / rho;
  W[0] = rho;
  double u2 = 0.0;
#pragma unroll
  for (int d = 0; d < ND; ++d) {
    W[1 + d] = U[1 + d] * ir;
    u2 += W[1 + d] * W[1 + d];
  }
  W[1 + ND] = eos_pressure(P, rho, U[1 + ND] - 0.5 * rho * u2);
  for (int s = 2 + ND; s < nv; ++s) W[s] = U[s] * ir;
}

template <int ND>
__device__ __forceinline__ void prim_to_cons(const Phys& P, int nv, const double* W, double* U) {
  const double rho = W[0];
  U[0] = rho;
  double u2 = 0.0;
#pragma unroll
  for (int d = 0; d < ND; ++d) {
    U[1 + d] = rho * W[1 + d];
    u2 += W[1 + d] * W[1 + d];
  }
  U[1 + ND] = eos_energy(P, rho, W[1 + ND]) + 0.5 * rho * u2;
  for (int s = 2 + ND; s < nv; ++s) U[s] = rho * W[s];
}

// Analytic flux along dir from primitives W and the matching conserved U (Eq. 1).
template <int ND>
__device__ __forceinline__ void flux_along(int nv, int dir, const double* W, const double* U, double* F) {
  const double un = W[1 + dir];
  const double p = W[1 + ND];
  F[0] = U[0] * un;
#pragma unroll
  for (int d = 0; d < ND; ++d) F[1 + d] = U[1 + d] * un + (d == dir ? p : 0.0);
  F[1 + ND] = (U[1 + ND] + p) * un;
  for (int s = 2 + ND; s < nv; ++s) F[s] = U[s] * un;
}

// ---------------------------------------------------------------------------------------------
// Riemann flux across a face normal to dir between conserved states UL | UR (L197-L201; Toro 2009
// ch. 10; Davis wave speeds R14; ties R15).
// ---------------------------------------------------------------------------------------------
template <int ND, int NVA>
__device__ __forceinline__ void riemann_flux(const Phys& P, int nv, int dir, const double* UL, const double* UR, double* F) {
  double WL[NVA], WR[NVA], FL[NVA], FR[NVA];
  cons_to_prim<ND>(P, nv, UL, WL);
  cons_to_prim<ND>(P, nv, UR, WR);
  flux_along<ND>(nv, dir, WL, UL, FL);
  flux_along<ND>(nv, dir, WR, UR, FR);
  const double rL = WL[0], rR = WR[0], uL = WL[1 + dir], uR = WR[1 + dir], pL = WL[1 + ND], pR = WR[1 + ND];
  const double cL = eos_sound_speed(P, rL, pL), cR = eos_sound_speed(P, rR, pR);
  const double SL = fmin(uL - cL, uR - cR), SR = fmax(uL + cL, uR + cR);
  if (P.riemann == HX_RIEMANN_HLL) {
    if (SL >= 0.0) {
      for (int v = 0; v < nv; ++v) F[v] = FL[v];
    } else if (SR <= 0.0) {
      for (int v = 0; v < nv; ++v) F[v] = FR[v];
    } else {
      const double iw = 1.0 / (SR - SL);
      for (int v = 0; v < nv; ++v) F[v] = (SR * FL[v] - SL * FR[v] + SL * SR * (UR[v] - UL[v])) * iw;
    }
    return;
  }
  const double mL = rL * (SL - uL), mR = rR * (SR - uR);
  const double Ss = (pR - pL + uL * mL - uR * mR) / (mL - mR);
  const bool left = (Ss >= 0.0);
  if (SL >= 0.0) {
    for (int v = 0; v < nv; ++v) F[v] = FL[v];
  } else if (!left && SR <= 0.0) {
    for (int v = 0; v < nv; ++v) F[v] = FR[v];
  } else {
    const double* UK = left ? UL : UR;
    const double* WK = left ? WL : WR;
    const double* FK = left ? FL : FR;
    const double SK = left ? SL : SR, mK = left ? mL : mR, uK = left ? uL : uR, pK = left ? pL : pR, rK = left ? rL : rR;
    const double fac = mK / (SK - Ss);
    F[0] = FK[0] + SK * (fac - UK[0]);
#pragma unroll
    for (int d = 0; d < ND; ++d) F[1 + d] = FK[1 + d] + SK * (fac * (d == dir ? Ss : WK[1 + d]) - UK[1 + d]);
    F[1 + ND] = FK[1 + ND] + SK * (fac * (UK[1 + ND] / rK + (Ss - uK) * (Ss + pK / mK)) - UK[1 + ND]);
    for (int s = 2 + ND; s < nv; ++s) F[s] = FK[s] + SK * (fac * WK[s] - UK[s]);
  }
}

// ---------------------------------------------------------------------------------------------
// Internal-energy monitoring (Eq. 10-12; R29).  Per face, next to the Riemann flux: the advective
// flux of e = (mass flux) x (e / rho of the upwind predicted state) and the face velocity = contact speed S* of the
// same Riemann problem (u_L or u_R when the whole fan lies on one side).
// ---------------------------------------------------------------------------------------------
template <int ND, int NVA>
__device__ __forceinline__ void monitor_face(const Phys& P, int nv, int dir, const double* UL, const double* UR, double fmass, double& phi,
                                             double& uface) {
  double WL[NVA], WR[NVA];
  cons_to_prim<ND>(P, nv, UL, WL);
  cons_to_prim<ND>(P, nv, UR, WR);
  const double rL = WL[0], rR = WR[0], uL = WL[1 + dir], uR = WR[1 + dir], pL = WL[1 + ND], pR = WR[1 + ND];
  const double cL = eos_sound_speed(P, rL, pL), cR = eos_sound_speed(P, rR, pR);
  const double SL = fmin(uL - cL, uR - cR), SR = fmax(uL + cL, uR + cR);
  if (SL >= 0.0) {
    uface = uL;
  } else if (SR <= 0.0) {
    uface = uR;
  } else {
    const double mL = rL * (SL - uL), mR = rR * (SR - uR);
    uface = (pR - pL + uL * mL - uR * mR) / (mL - mR);
  }
  const bool left = fmass >= 0.0;
  const double* UK = left ? UL : UR;
  const double* WK = left ? WL : WR;
  double u2 = 0.0;
#pragma unroll
  for (int d = 0; d < ND; ++d) u2 += WK[1 + d] * WK[1 + d];
  phi = fmass * (UK[1 + ND] - 0.5 * WK[0] * u2) / WK[0];
}

// Eq. 11-12: blend of the internal energy e1 (from the total-energy update) and e2 (from Eq. 10); returns the new e.
__device__ __forceinline__ double monitor_blend(double eps, double en, double e1, double e2, double ek) {
  const double lim = eps * ek;
  double alpha;
  if (e1 >= lim) alpha = 1.0;
  else if (e1 > 0.1 * lim) alpha = (e1 / lim) * (e1 / lim);
  else alpha = 0.0;
  return en + alpha * (e1 - en) + (1.0 - alpha) * (e2 - en);
}

// ---------------------------------------------------------------------------------------------
// Reductions
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// Block-wide max of a non-negative double, one atomicMax per block on its bit pattern (positive
// IEEE doubles order like unsigned integers).  All threads of the block must call it.
__device__ __forceinline__ void block_rate_max(double rate, unsigned long long* out) {
  __shared__ double s_part[32];
  const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
  const int nthreads = blockDim.x * blockDim.y * blockDim.z;
  rate = warp_max(rate);
  if ((tid & 31) == 0) s_part[tid >> 5] = rate;
  __syncthreads();
  if (tid < 32) {
    double v = (tid < (nthreads + 31) / 32) ? s_part[tid] : 0.0;
    v = warp_max(v);
    if (tid == 0) atomicMax(out, (unsigned long long)__double_as_longlong(v));
  }
}

}  // namespace hx

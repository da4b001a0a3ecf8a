// ox_oracle.cpp -- CPU ORACLE (test infrastructure, not the product) for the unsplit
// MUSCL-Hancock / Godunov finite-volume hydro step of HERACLES++ (arxiv 2503.04428).
//
// Plain, slow, whole-array passes in fp64, following PAPER.md in the paper's order:
//   O0 ghost fill      : Sect. 3.2 "periodic, null gradient, reflective"
//   O1 cons -> prim    : Eq. 1 + ideal-gas EOS Eq. 5, or gas + radiation Eq. 6-7 (L44-L57, L83-L102)
//   O2 limited slopes  : Eq. 17, limiters Minmod / Van Leer / Van Albada (+ MC)  (L184-L189)
//   O3 face states     : Eq. 17
//   O4 Hancock half step: Eq. 18, multi-D as Toro Sect. 16.5 (unsplit)           (L191-L195)
//   O5 Riemann flux    : HLL / HLLC (Toro 2009)                                  (L197-L201)
//   O6 update + sources: Eq. 19, spherical sources Eq. 13-16, gravity Eq. 1b-1c, 2, 3, 4 (self-gravity),
//                        internal-energy monitoring Eq. 10-12
//   O7 CFL time step   : sum form (reading R2 in DESIGN.md)
// Where the paper is silent or garbled the readings R1-R29 listed in DESIGN.md apply.
//
// A second, deliberately naive per-cell evaluation (ox_cell_update) is written separately
// from the same passages with boundary conditions applied by index mapping; tests compare
// the two (pin P11) and use the per-cell form to check sampled cells of full-size GPU runs.
//
// Shares NO code with the CUDA path.  Compile: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC.
// Pins: tests/test_oracle_*.py (exact Sod solution, convergence orders, uniform state,
// conservation, F(U,U)=F(U), stationary contact, symmetry, angular momentum, free fall,
// spherical 1-D/3-D reduction, Sedov similarity radius centred and off-centre, brute force, EOS round trip / Eq. 7
// against the adiabatic derivative / limits, self-gravity closed forms).  Every function is pinned: none is
// "parity unpinned".
#include "ox.h"

#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstring>
#include <limits>
#include <new>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int NG = 2;       // ghost layers per face in active directions
constexpr int NVMAX = 16;   // 2 + 3 + up to 11 passive scalars
constexpr int NFMAX = NVMAX + 2;   // a face flux vector: the fields + the advective flux of e and the face velocity (monitoring, R29)

inline bool is_reflecting(int bc) { return bc == OX_BC_REFLECTING || bc == OX_BC_WEDGE; }

}  // namespace

struct ox_handle {
  ox_config c;
  int nvar;
  int ng[3];               // NG if the direction is active else 0
  int np[3];               // padded sizes
  size_t ncp;              // padded cells
  std::vector<double> xf[3];  // padded face coordinates, xf[d][idx + ng[d]] = minus face of cell idx
  std::vector<double> U;      // conserved state, [nvar][np2][np1][np0]
  std::vector<double> gself;  // OX_GRAV_SELF: g_r at the centres of the interior radial cells, for the state in U
  double gself_mtot = 0.0;    // ... and G times the whole enclosed mass (cells beyond the outer radius)
  bool gself_dirty = true;

  size_t cell(int i, int j, int k) const {
    return ((size_t)(k + ng[2]) * np[1] + (size_t)(j + ng[1])) * np[0] + (size_t)(i + ng[0]);
  }
  double fm(int d, int idx) const { return xf[d][idx + ng[d]]; }       // minus face
  double fp(int d, int idx) const { return xf[d][idx + ng[d] + 1]; }   // plus face
  double xc(int d, int idx) const { return 0.5 * (fm(d, idx) + fp(d, idx)); }  // R6: arithmetic midpoint
  double width(int d, int idx) const { return fp(d, idx) - fm(d, idx); }
};

namespace {

// ----------------------------------------------------------------------------------------
// Geometry ("surface elements (dS) and volumes (dV) of cells are computed
// based on the chosen geometry").  dS[d][0] = minus face, dS[d][1] = plus face.
// ----------------------------------------------------------------------------------------
void cell_geometry(const ox_handle* h, int i, int j, int k, double& dV, double dS[3][2]) {
  const int id[3] = {i, j, k};
  double lo[3], hi[3];
  for (int d = 0; d < 3; ++d) {
    lo[d] = h->fm(d, id[d]);
    hi[d] = h->fp(d, id[d]);
  }
  if (h->c.coords == OX_CARTESIAN) {
    const double w0 = hi[0] - lo[0], w1 = hi[1] - lo[1], w2 = hi[2] - lo[2];
    dV = w0 * w1 * w2;
    dS[0][0] = dS[0][1] = w1 * w2;
    dS[1][0] = dS[1][1] = w0 * w2;
    dS[2][0] = dS[2][1] = w0 * w1;
  } else {
    const double rm = lo[0], rp = hi[0], tm = lo[1], tp = hi[1];
    const double dphi = hi[2] - lo[2];
    const double dcos = std::cos(tm) - std::cos(tp);
    const double r3 = (rp * rp * rp - rm * rm * rm) / 3.0;
    const double r2 = (rp * rp - rm * rm) / 2.0;
    dV = r3 * dcos * dphi;
    dS[0][0] = rm * rm * dcos * dphi;
    dS[0][1] = rp * rp * dcos * dphi;
    dS[1][0] = std::sin(tm) * r2 * dphi;
    dS[1][1] = std::sin(tp) * r2 * dphi;
    dS[2][0] = dS[2][1] = r2 * (tp - tm);
  }
}

// Gravitational acceleration component g_d seen by cell index idx along direction d.
// Uniform: Eq. 2 (acceleration vector, reading R12).  Point mass: Eq. 3, -GM/r_c^2 on d = 0.
// Ghost cells behind a reflecting boundary carry the mirror image of the field (reading R25),
// ghost cells behind a periodic boundary the wrapped value.
double gravity_raw(const ox_handle* h, int d, int idx) {
  if (h->c.gravity == OX_GRAV_UNIFORM) return h->c.g[d];
  if (h->c.gravity == OX_GRAV_POINT_MASS) {
    if (d != 0) return 0.0;
    const double rc = h->xc(0, idx);
    return -h->c.GM / (rc * rc);
  }
  if (h->c.gravity == OX_GRAV_SELF) {   // Eq. 4 with the table refresh_self_gravity() made for the current state
    if (d != 0) return 0.0;
    if (idx >= 0 && idx < h->c.n[0]) return h->gself[idx];
    const double rc = h->xc(0, idx);
    return -(idx < 0 ? h->c.GM : h->gself_mtot) / (rc * rc);   // inside r_min: the central mass only; outside r_max: everything
  }
  return 0.0;
}

// Eq. 4 (L73-L77): g(r, t) = -G M(r, t) / r^2 e_r, "M(r,t) the total mass within the sphere of radius r", "in the
// approximation of a spherically symmetric matter distribution".  Reading R28: at the centre r_c of radial cell i
//   M = M_c + (4 pi / dOmega) [ sum_{i' < i} m_i' + m_i (r_c^3 - r_-^3) / (r_+^3 - r_-^3) ],   m_i = sum_{j,k} rho dV,
// dOmega the solid angle of the grid (the wedge stands for the whole sphere), the shell of cell i counted up to r_c
// by volume; the field of the state at the START of a step is used for the whole step.
void refresh_self_gravity(ox_handle* h) {
  if (h->c.gravity != OX_GRAV_SELF || !h->gself_dirty) return;
  const ox_config& c = h->c;
  const int n0 = c.n[0];
  std::vector<double> m(n0, 0.0);
  for (int k = 0; k < c.n[2]; ++k)
    for (int j = 0; j < c.n[1]; ++j)
      for (int i = 0; i < n0; ++i) {
        double dV, dS[3][2];
        cell_geometry(h, i, j, k, dV, dS);
        m[i] += h->U[h->cell(i, j, k)] * dV;
      }
  const double PI = 3.14159265358979323846;
  const double domega = (std::cos(h->fm(1, 0)) - std::cos(h->fp(1, c.n[1] - 1))) * (h->fp(2, c.n[2] - 1) - h->fm(2, 0));
  const double scale = c.G * 4.0 * PI / domega;
  h->gself.assign(n0, 0.0);
  double below = 0.0;
  for (int i = 0; i < n0; ++i) {
    const double rm = h->fm(0, i), rp = h->fp(0, i), rc = h->xc(0, i);
    const double frac = (rc * rc * rc - rm * rm * rm) / (rp * rp * rp - rm * rm * rm);
    h->gself[i] = -(c.GM + scale * (below + m[i] * frac)) / (rc * rc);
    below += m[i];
  }
  h->gself_mtot = c.GM + scale * below;
  h->gself_dirty = false;
}
double gravity(const ox_handle* h, int d, int idx) {
  if (h->c.gravity == OX_GRAV_NONE || d >= h->c.ndim) return 0.0;
  const int n = h->c.n[d];
  if (idx < 0) {
    if (is_reflecting(h->c.bc_lo[d])) return -gravity_raw(h, d, -1 - idx);
    if (h->c.bc_lo[d] == OX_BC_PERIODIC) return gravity_raw(h, d, idx + n);
  } else if (idx >= n) {
    if (is_reflecting(h->c.bc_hi[d])) return -gravity_raw(h, d, 2 * n - 1 - idx);
    if (h->c.bc_hi[d] == OX_BC_PERIODIC) return gravity_raw(h, d, idx - n);
  }
  return gravity_raw(h, d, idx);
}

// ----------------------------------------------------------------------------------------
// Pointwise physics
// ----------------------------------------------------------------------------------------
// Equation of state.  Ideal gas (Eq. 5): P = (gamma-1) e, c_s = sqrt(gamma P / rho).  Gas + radiation (Eq. 6-7):
//   e = rho R T / (gamma-1) + a_r T^4,   P = rho R T + a_r T^4 / 3   (R = k_b / mu),
//   c_s^2 = [gamma/(gamma-1) + 20 alpha + 16 alpha^2] / [1/(gamma-1) + 12 alpha] * P_g / rho,  alpha = P_r / P_g;
// "the pressure cannot be computed directly from the internal energy, so we first need to determine the
// temperature ... using the internal energy equation 6a and a Newton-Raphson approach" (L102).  The same solve
// gives T from P when a primitive state is turned into a conserved one.
struct Eos {
  int kind;
  double gamma, R, ar;
  Eos(double g) : kind(OX_EOS_IDEAL), gamma(g), R(0.0), ar(0.0) {}   // ideal gas from its adiabatic index
  Eos(int k, double g, double r, double a) : kind(k), gamma(g), R(r), ar(a) {}
};

// Positive root of lin*T + quart*T^4 = rhs (lin, quart > 0).  The start min(rhs/lin, (rhs/quart)^(1/4)) lies at or
// above the root of this convex increasing function, so Newton-Raphson descends monotonically onto it.
double newton_T(double lin, double quart, double rhs) {
  if (!(rhs > 0.0)) return rhs / lin;   // non-physical input: hand back a non-positive T, the caller's P > 0 check reports it
  double T = std::min(rhs / lin, std::pow(rhs / quart, 0.25));
  // stop when the correction is a few ulp (reading R27; a bound below the rounding unit would never be met and
  // the loop would always run to its cap); the iteration converges quadratically, ~5-9 steps (L102: "approximately ten")
  for (int it = 0; it < 60; ++it) {
    const double T3 = T * T * T;
    const double f = lin * T + quart * T3 * T - rhs;
    const double dT = f / (lin + 4.0 * quart * T3);
    T -= dT;
    if (std::fabs(dT) <= 1e-15 * T) break;
  }
  return T;
}

double eos_pressure(const Eos& q, double rho, double e) {   // P(rho, e)
  if (q.kind == OX_EOS_IDEAL) return (q.gamma - 1.0) * e;
  const double T = newton_T(rho * q.R / (q.gamma - 1.0), q.ar, e);
  return rho * q.R * T + q.ar * T * T * T * T / 3.0;
}

double eos_energy(const Eos& q, double rho, double P) {     // e(rho, P)
  if (q.kind == OX_EOS_IDEAL) return P / (q.gamma - 1.0);
  const double T = newton_T(rho * q.R, q.ar / 3.0, P);
  return rho * q.R * T / (q.gamma - 1.0) + q.ar * T * T * T * T;
}

double eos_sound_speed(const Eos& q, double rho, double P) {   // c_s(rho, P)
  if (q.kind == OX_EOS_IDEAL) return std::sqrt(q.gamma * P / rho);
  const double T = newton_T(rho * q.R, q.ar / 3.0, P);
  const double Pg = rho * q.R * T, Pr = q.ar * T * T * T * T / 3.0;
  const double al = Pr / Pg;
  return std::sqrt((q.gamma / (q.gamma - 1.0) + 20.0 * al + 16.0 * al * al) / (1.0 / (q.gamma - 1.0) + 12.0 * al) * Pg / rho);
}

Eos eos_of(const ox_config& c) { return Eos(c.eos, c.gamma, c.eos_R, c.eos_ar); }

// O1 (Eq. 1, Eq. 5 / 6): rho; u_d = m_d/rho; e = E - rho|u|^2/2; P = P(rho, e); f_s = (rho f_s)/rho
void cons_to_prim(const Eos& eos, int ndim, int nvar, const double* U, double* W) {
  const double rho = U[0];
  W[0] = rho;
  double u2 = 0.0;
  for (int d = 0; d < ndim; ++d) {
    W[1 + d] = U[1 + d] / rho;
    u2 += W[1 + d] * W[1 + d];
  }
  const double e = U[1 + ndim] - 0.5 * rho * u2;
  W[1 + ndim] = eos_pressure(eos, rho, e);
  for (int s = 2 + ndim; s < nvar; ++s) W[s] = U[s] / rho;
}

void prim_to_cons(const Eos& eos, int ndim, int nvar, const double* W, double* U) {
  const double rho = W[0];
  U[0] = rho;
  double u2 = 0.0;
  for (int d = 0; d < ndim; ++d) {
    U[1 + d] = rho * W[1 + d];
    u2 += W[1 + d] * W[1 + d];
  }
  U[1 + ndim] = eos_energy(eos, rho, W[1 + ndim]) + 0.5 * rho * u2;
  for (int s = 2 + ndim; s < nvar; ++s) U[s] = rho * W[s];
}

// Analytic flux in direction dir from primitives (Eq. 1):
// (rho u_n, rho u_n u_d + P delta_{d,dir}, (E+P) u_n, rho f_s u_n)
void flux_from_prim(const Eos& eos, int ndim, int nvar, int dir, const double* W, double* F) {
  double U[NVMAX];
  prim_to_cons(eos, ndim, nvar, W, U);
  const double un = W[1 + dir];
  const double P = W[1 + ndim];
  F[0] = U[0] * un;
  for (int d = 0; d < ndim; ++d) F[1 + d] = U[1 + d] * un + (d == dir ? P : 0.0);
  F[1 + ndim] = (U[1 + ndim] + P) * un;
  for (int s = 2 + ndim; s < nvar; ++s) F[s] = U[s] * un;
}

// O2 limiters (Eq. 17; R3-R5): a = backward gradient, b = forward gradient
double limiter(int lim, double a, double b) {
  if (lim == OX_LIM_NONE) return 0.0;
  if (a * b <= 0.0) return 0.0;
  const double sa = (a > 0.0) ? 1.0 : -1.0;
  switch (lim) {
    case OX_LIM_MINMOD:
      return sa * std::min(std::fabs(a), std::fabs(b));
    case OX_LIM_VANLEER:
      return 2.0 * a * b / (a + b);
    case OX_LIM_VANALBADA:
      return a * b * (a + b) / (a * a + b * b);
    case OX_LIM_MC:
      return sa * std::min(std::min(2.0 * std::fabs(a), 2.0 * std::fabs(b)), 0.5 * std::fabs(a + b));
    default:
      return 0.0;
  }
}

// O5 Riemann flux between conserved states UL | UR across a face normal to dir (Toro 2009,
// ch. 10; wave-speed estimates of Davis, reading R14; ties per R15).
void riemann_flux_core(int solver, const Eos& eos, int ndim, int nvar, int dir, const double* UL, const double* UR,
                       double* F) {
  double WL[NVMAX], WR[NVMAX], FL[NVMAX], FR[NVMAX];
  cons_to_prim(eos, ndim, nvar, UL, WL);
  cons_to_prim(eos, ndim, nvar, UR, WR);
  flux_from_prim(eos, ndim, nvar, dir, WL, FL);
  flux_from_prim(eos, ndim, nvar, dir, WR, FR);
  const int ie = 1 + ndim;
  const double rL = WL[0], rR = WR[0], uL = WL[1 + dir], uR = WR[1 + dir], PL = WL[ie], PR = WR[ie];
  const double cL = eos_sound_speed(eos, rL, PL), cR = eos_sound_speed(eos, rR, PR);
  const double SL = std::min(uL - cL, uR - cR);
  const double SR = std::max(uL + cL, uR + cR);
  if (solver == OX_RIEMANN_HLL) {
    if (SL >= 0.0) {
      for (int v = 0; v < nvar; ++v) F[v] = FL[v];
    } else if (SR <= 0.0) {
      for (int v = 0; v < nvar; ++v) F[v] = FR[v];
    } else {
      for (int v = 0; v < nvar; ++v) F[v] = (SR * FL[v] - SL * FR[v] + SL * SR * (UR[v] - UL[v])) / (SR - SL);
    }
    return;
  }
  // HLLC
  const double Sstar =
      (PR - PL + rL * uL * (SL - uL) - rR * uR * (SR - uR)) / (rL * (SL - uL) - rR * (SR - uR));
  auto star_state = [&](const double* UK, const double* WK, double SK, double* Us) {
    const double rK = WK[0], uK = WK[1 + dir], PK = WK[ie];
    const double fac = rK * (SK - uK) / (SK - Sstar);
    Us[0] = fac;
    for (int d = 0; d < ndim; ++d) Us[1 + d] = fac * (d == dir ? Sstar : WK[1 + d]);
    Us[ie] = fac * (UK[ie] / rK + (Sstar - uK) * (Sstar + PK / (rK * (SK - uK))));
    for (int s = 2 + ndim; s < nvar; ++s) Us[s] = fac * WK[s];
  };
  double Us[NVMAX];
  if (SL >= 0.0) {
    for (int v = 0; v < nvar; ++v) F[v] = FL[v];
  } else if (Sstar >= 0.0) {
    star_state(UL, WL, SL, Us);
    for (int v = 0; v < nvar; ++v) F[v] = FL[v] + SL * (Us[v] - UL[v]);
  } else if (SR > 0.0) {
    star_state(UR, WR, SR, Us);
    for (int v = 0; v < nvar; ++v) F[v] = FR[v] + SR * (Us[v] - UR[v]);
  } else {
    for (int v = 0; v < nvar; ++v) F[v] = FR[v];
  }
}

// Internal-energy monitoring (Eq. 10; reading R29): what the second energy equation
//   de/dt + div(u e) + P div u = 0
// needs from a face: the advective flux of e, taken as (mass flux) x (e/rho of the upwind predicted state), and the
// face velocity "from the standard hydrodynamical step", taken as the contact speed S* of the same Riemann problem
// (Toro Eq. 10.37 with the wave speeds of R14; the left / right velocity when the whole fan lies on one side).
void monitor_face(const Eos& eos, int ndim, int nvar, int dir, const double* UL, const double* UR, double Fmass, double& phi,
                  double& uface) {
  double WL[NVMAX], WR[NVMAX];
  cons_to_prim(eos, ndim, nvar, UL, WL);
  cons_to_prim(eos, ndim, nvar, UR, WR);
  const int ie = 1 + ndim;
  const double rL = WL[0], rR = WR[0], uL = WL[1 + dir], uR = WR[1 + dir], PL = WL[ie], PR = WR[ie];
  const double cL = eos_sound_speed(eos, rL, PL), cR = eos_sound_speed(eos, rR, PR);
  const double SL = std::min(uL - cL, uR - cR), SR = std::max(uL + cL, uR + cR);
  if (SL >= 0.0) uface = uL;
  else if (SR <= 0.0) uface = uR;
  else {
    const double mL = rL * (SL - uL), mR = rR * (SR - uR);
    uface = (PR - PL + uL * mL - uR * mR) / (mL - mR);
  }
  const double* UK = (Fmass >= 0.0) ? UL : UR;
  const double* WK = (Fmass >= 0.0) ? WL : WR;
  double u2 = 0.0;
  for (int d = 0; d < ndim; ++d) u2 += WK[1 + d] * WK[1 + d];
  phi = Fmass * (UK[ie] - 0.5 * WK[0] * u2) / WK[0];
}

// F[0..nvar-1]: Riemann flux; F[nvar]: advective flux of the internal energy; F[nvar+1]: face velocity (monitoring)
void riemann_flux(int solver, const Eos& eos, int ndim, int nvar, int dir, const double* UL, const double* UR,
                  double* F) {
  riemann_flux_core(solver, eos, ndim, nvar, dir, UL, UR, F);
  monitor_face(eos, ndim, nvar, dir, UL, UR, F[0], F[nvar], F[nvar + 1]);
}

// Cell-centred geometric source of the predictor in spherical coordinates (O4, reading R8):
// the cell-centred limit of the O6 sources.  Velocities of inactive directions are zero.
void spherical_G(const ox_handle* h, int i, int j, const double* W, double dV, const double dS[3][2], double* G) {
  const int ndim = h->c.ndim;
  const double rho = W[0], ur = W[1], ut = (ndim >= 2) ? W[2] : 0.0, up = (ndim >= 3) ? W[3] : 0.0;
  const double P = W[1 + ndim];
  const double rm = h->fm(0, i), rp = h->fp(0, i);
  const double A_r = (rp - rm) * (dS[0][1] + dS[0][0]) / ((rp + rm) * dV);
  G[0] = (rho * ut * ut + rho * up * up + 2.0 * P) * (dS[0][1] - dS[0][0]) / (2.0 * dV);
  G[1] = G[2] = 0.0;
  if (ndim >= 2) G[1] = -rho * ut * ur * A_r + (rho * up * up + P) * (dS[1][1] - dS[1][0]) / dV;
  if (ndim >= 3) {
    const double sm = std::sin(h->fm(1, j)), sp = std::sin(h->fp(1, j));
    const double A_t = (sp - sm) * (dS[1][1] + dS[1][0]) / ((sp + sm) * dV);
    G[2] = -rho * up * ur * A_r - rho * up * ut * A_t;
  }
}

// Spherical momentum sources of the update from the face Riemann fluxes (O6; Eq. 14-16, R9-R11).
// Fm[d], Fp[d] = Riemann flux vectors through the minus/plus face of direction d (active d only);
// Pbar replaces the normal momentum flux through the faces of inactive angular directions.
void spherical_S(const ox_handle* h, int i, int j, const double* const Fm[3], const double* const Fp[3],
                 double Pbar, double dV, const double dS[3][2], double* S) {
  const int ndim = h->c.ndim;
  const double rm = h->fm(0, i), rp = h->fp(0, i);
  const double Ftt_m = (ndim >= 2) ? Fm[1][2] : Pbar, Ftt_p = (ndim >= 2) ? Fp[1][2] : Pbar;
  const double Fpp_m = (ndim >= 3) ? Fm[2][3] : Pbar, Fpp_p = (ndim >= 3) ? Fp[2][3] : Pbar;
  S[0] = (0.5 * (Ftt_m + Ftt_p) + 0.5 * (Fpp_m + Fpp_p)) * (dS[0][1] - dS[0][0]) / (2.0 * dV);
  S[1] = S[2] = 0.0;
  const double cr = (rp - rm) / ((rp + rm) * dV);
  if (ndim >= 2)
    S[1] = -cr * (Fp[0][2] * dS[0][1] + Fm[0][2] * dS[0][0]) + 0.5 * (Fpp_m + Fpp_p) * (dS[1][1] - dS[1][0]) / dV;
  if (ndim >= 3) {
    const double sm = std::sin(h->fm(1, j)), sp = std::sin(h->fp(1, j));
    const double ct = (sp - sm) / ((sp + sm) * dV);
    S[2] = -cr * (Fp[0][3] * dS[0][1] + Fm[0][3] * dS[0][0]) - ct * (Fp[1][3] * dS[1][1] + Fm[1][3] * dS[1][0]);
  }
}

// O2-O4 for one cell given the primitives of the cell and of its face neighbours:
// Wn[d][0] = neighbour at -1, Wn[d][1] = neighbour at +1 in direction d.
// Outputs the predicted conservative face states Um[d], Up[d] and the pressure Pbar of the
// cell-centred predicted state U^n + dU.
void predictor(const ox_handle* h, int i, int j, int k, double dt, const double* W, const double Wn[3][2][NVMAX],
               double Um[3][NVMAX], double Up[3][NVMAX], double& Pbar) {
  const ox_config& c = h->c;
  const int ndim = c.ndim, nvar = h->nvar;
  const int id[3] = {i, j, k};
  double U[NVMAX];
  prim_to_cons(eos_of(c), ndim, nvar, W, U);
  if (c.limiter == OX_LIM_NONE) {  // R19: first-order Godunov, no predictor
    for (int d = 0; d < ndim; ++d)
      for (int v = 0; v < nvar; ++v) Um[d][v] = Up[d][v] = U[v];
    Pbar = W[1 + ndim];
    return;
  }
  double dV, dS[3][2];
  cell_geometry(h, i, j, k, dV, dS);
  double Wm[3][NVMAX], Wp[3][NVMAX];
  double dU[NVMAX];
  for (int v = 0; v < nvar; ++v) dU[v] = 0.0;
  for (int d = 0; d < ndim; ++d) {
    const double xm = h->xc(d, id[d] - 1), x0 = h->xc(d, id[d]), xp = h->xc(d, id[d] + 1);
    const double del = h->width(d, id[d]);
    for (int v = 0; v < nvar; ++v) {
      const double a = (W[v] - Wn[d][0][v]) / (x0 - xm);   // O2, R5
      const double b = (Wn[d][1][v] - W[v]) / (xp - x0);
      const double sig = limiter(c.limiter, a, b);
      Wm[d][v] = W[v] - 0.5 * del * sig;                   // O3, Eq. 17
      Wp[d][v] = W[v] + 0.5 * del * sig;
    }
    double Fm[NVMAX], Fp[NVMAX];
    flux_from_prim(eos_of(c), ndim, nvar, d, Wm[d], Fm);
    flux_from_prim(eos_of(c), ndim, nvar, d, Wp[d], Fp);
    for (int v = 0; v < nvar; ++v) dU[v] += (Fm[v] * dS[d][0] - Fp[v] * dS[d][1]) / dV;  // O4, Eq. 18
  }
  if (c.coords == OX_SPHERICAL) {
    double G[3];
    spherical_G(h, i, j, W, dV, dS, G);
    for (int d = 0; d < ndim; ++d) dU[1 + d] += G[d];
  }
  for (int d = 0; d < ndim; ++d) {  // S_g (R12, R13)
    const double gd = gravity(h, d, id[d]);
    dU[1 + d] += W[0] * gd;
    dU[1 + ndim] += U[1 + d] * gd;
  }
  for (int v = 0; v < nvar; ++v) dU[v] *= 0.5 * dt;
  for (int d = 0; d < ndim; ++d) {
    prim_to_cons(eos_of(c), ndim, nvar, Wm[d], Um[d]);
    prim_to_cons(eos_of(c), ndim, nvar, Wp[d], Up[d]);
    for (int v = 0; v < nvar; ++v) {
      Um[d][v] += dU[v];
      Up[d][v] += dU[v];
    }
  }
  double Uc[NVMAX], Wc[NVMAX];
  for (int v = 0; v < nvar; ++v) Uc[v] = U[v] + dU[v];
  cons_to_prim(eos_of(c), ndim, nvar, Uc, Wc);
  Pbar = Wc[1 + ndim];
}

// O6 for one cell from its six face fluxes.
void update_cell(const ox_handle* h, int i, int j, int k, double dt, const double* Un, const double* const Fm[3],
                 const double* const Fp[3], double Pbar, double* Unew) {
  const ox_config& c = h->c;
  const int ndim = c.ndim, nvar = h->nvar;
  const int id[3] = {i, j, k};
  double dV, dS[3][2];
  cell_geometry(h, i, j, k, dV, dS);
  for (int v = 0; v < nvar; ++v) {
    double acc = 0.0;
    for (int d = 0; d < ndim; ++d) acc += Fm[d][v] * dS[d][0] - Fp[d][v] * dS[d][1];
    Unew[v] = Un[v] + (dt / dV) * acc;  // Eq. 19
  }
  if (c.coords == OX_SPHERICAL) {
    double S[3];
    spherical_S(h, i, j, Fm, Fp, Pbar, dV, dS, S);
    for (int d = 0; d < ndim; ++d) Unew[1 + d] += dt * S[d];
  }
  if (c.gravity != OX_GRAV_NONE) {  // time-centred (R13)
    for (int d = 0; d < ndim; ++d) {
      const double gd = gravity(h, d, id[d]);
      const double mstar = Unew[1 + d];
      Unew[1 + d] = mstar + dt * 0.5 * (Un[0] + Unew[0]) * gd;
      Unew[1 + ndim] += dt * 0.5 * (Un[1 + d] + Unew[1 + d]) * gd;
    }
  }
  if (c.emon_eps > 0.0) {   // monitoring of the internal energy in highly supersonic regions (Eq. 10-12, reading R29)
    const int ie = 1 + ndim;
    double Wn[NVMAX];
    cons_to_prim(eos_of(c), ndim, nvar, Un, Wn);
    double kn = 0.0, k1 = 0.0;
    for (int d = 0; d < ndim; ++d) {
      kn += Un[1 + d] * Un[1 + d];
      k1 += Unew[1 + d] * Unew[1 + d];
    }
    const double en = Un[ie] - 0.5 * kn / Un[0];            // e^n
    const double ek = 0.5 * k1 / Unew[0];                   // kinetic energy of the new state
    const double e1 = Unew[ie] - ek;                        // e^n + delta^1 e: from the total-energy equation (Eq. 1c)
    double adv = 0.0, divu = 0.0;                           // Eq. 10: -div(u e) and div u, finite-volume form
    for (int d = 0; d < ndim; ++d) {
      adv += Fm[d][nvar] * dS[d][0] - Fp[d][nvar] * dS[d][1];
      divu += Fp[d][nvar + 1] * dS[d][1] - Fm[d][nvar + 1] * dS[d][0];
    }
    const double e2 = en + (dt / dV) * (adv - Wn[ie] * divu);   // e^n + delta^2 e, pressure of the old state
    const double lim = c.emon_eps * ek;                     // Eq. 12
    double alpha;
    if (e1 >= lim) alpha = 1.0;
    else if (e1 > 0.1 * lim) alpha = (e1 / lim) * (e1 / lim);
    else alpha = 0.0;
    const double enew = en + alpha * (e1 - en) + (1.0 - alpha) * (e2 - en);   // Eq. 11
    Unew[ie] = ek + enew;
  }
}

// ----------------------------------------------------------------------------------------
// O0 ghost fill on the stored array: directions 0,1,2 in order, each pass spanning the
// full padded extent of the other directions (so edges and corners are defined).
// ----------------------------------------------------------------------------------------
void fill_ghosts(ox_handle* h, std::vector<double>& U) {
  const ox_config& c = h->c;
  for (int d = 0; d < c.ndim; ++d) {
    const int n = c.n[d];
    int lo[3], hi[3];
    for (int e = 0; e < 3; ++e) {
      lo[e] = -h->ng[e];
      hi[e] = c.n[e] + h->ng[e];
    }
    lo[d] = 0;
    hi[d] = 1;  // iterate the transverse extent only
    for (int v = 0; v < h->nvar; ++v) {
      double* Uv = &U[(size_t)v * h->ncp];
      const double flip = (v == 1 + d) ? -1.0 : 1.0;
      for (int k = lo[2]; k < hi[2]; ++k)
        for (int j = lo[1]; j < hi[1]; ++j)
          for (int i = lo[0]; i < hi[0]; ++i) {
            int id[3] = {i, j, k};
            for (int g = 1; g <= NG; ++g) {
              int src, dst;
              double s;
              // low side
              dst = -g;
              if (c.bc_lo[d] == OX_BC_PERIODIC) { src = n - g; s = 1.0; }
              else if (c.bc_lo[d] == OX_BC_TRANSMISSIVE) { src = 0; s = 1.0; }
              else { src = g - 1; s = flip; }
              id[d] = src; const double a = Uv[h->cell(id[0], id[1], id[2])];
              id[d] = dst; Uv[h->cell(id[0], id[1], id[2])] = s * a;
              // high side
              dst = n - 1 + g;
              if (c.bc_hi[d] == OX_BC_PERIODIC) { src = g - 1; s = 1.0; }
              else if (c.bc_hi[d] == OX_BC_TRANSMISSIVE) { src = n - 1; s = 1.0; }
              else { src = n - g; s = flip; }
              id[d] = src; const double b = Uv[h->cell(id[0], id[1], id[2])];
              id[d] = dst; Uv[h->cell(id[0], id[1], id[2])] = s * b;
            }
          }
    }
  }
}

// Boundary conditions by index mapping (used only by the naive per-cell evaluation).
// Returns the interior index that ghost index idx of direction d copies, and multiplies
// *sign by -1 when a reflecting boundary is crossed.
int map_index(const ox_handle* h, int d, int idx, double* sign) {
  const int n = h->c.n[d];
  if (idx < 0) {
    if (h->c.bc_lo[d] == OX_BC_PERIODIC) return idx + n;
    if (h->c.bc_lo[d] == OX_BC_TRANSMISSIVE) return 0;
    *sign = -*sign;
    return -1 - idx;
  }
  if (idx >= n) {
    if (h->c.bc_hi[d] == OX_BC_PERIODIC) return idx - n;
    if (h->c.bc_hi[d] == OX_BC_TRANSMISSIVE) return n - 1;
    *sign = -*sign;
    return 2 * n - 1 - idx;
  }
  return idx;
}

void naive_get_U(const ox_handle* h, int i, int j, int k, double* U) {
  const int id[3] = {i, j, k};
  int src[3];
  double sgn[3] = {1.0, 1.0, 1.0};
  for (int d = 0; d < 3; ++d) src[d] = (d < h->c.ndim) ? map_index(h, d, id[d], &sgn[d]) : 0;
  const size_t cidx = h->cell(src[0], src[1], src[2]);
  for (int v = 0; v < h->nvar; ++v) U[v] = h->U[(size_t)v * h->ncp + cidx];
  for (int d = 0; d < h->c.ndim; ++d) U[1 + d] *= sgn[d];
}

void naive_get_W(const ox_handle* h, int i, int j, int k, double* W) {
  double U[NVMAX];
  naive_get_U(h, i, j, k, U);
  cons_to_prim(eos_of(h->c), h->c.ndim, h->nvar, U, W);
}

void naive_predict(const ox_handle* h, int i, int j, int k, double dt, double Um[3][NVMAX], double Up[3][NVMAX],
                   double& Pbar) {
  double W[NVMAX], Wn[3][2][NVMAX];
  naive_get_W(h, i, j, k, W);
  for (int d = 0; d < h->c.ndim; ++d) {
    int a[3] = {i, j, k}, b[3] = {i, j, k};
    a[d] -= 1;
    b[d] += 1;
    naive_get_W(h, a[0], a[1], a[2], Wn[d][0]);
    naive_get_W(h, b[0], b[1], b[2], Wn[d][1]);
  }
  predictor(h, i, j, k, dt, W, Wn, Um, Up, Pbar);
}

// Riemann flux through the minus face of cell (i,j,k) in direction d.
void naive_face_flux(const ox_handle* h, int i, int j, int k, int d, double dt, double* F) {
  int a[3] = {i, j, k};
  a[d] -= 1;
  double UmL[3][NVMAX], UpL[3][NVMAX], UmR[3][NVMAX], UpR[3][NVMAX], pb;
  naive_predict(h, a[0], a[1], a[2], dt, UmL, UpL, pb);
  naive_predict(h, i, j, k, dt, UmR, UpR, pb);
  riemann_flux(h->c.riemann, eos_of(h->c), h->c.ndim, h->nvar, d, UpL[d], UmR[d], F);
}

int check_config(const ox_config* c) {
  if (!c) return OX_ERR_INVALID_ARG;
  if (c->ndim < 1 || c->ndim > 3) return OX_ERR_INVALID_ARG;
  if (c->coords != OX_CARTESIAN && c->coords != OX_SPHERICAL) return OX_ERR_INVALID_ARG;
  if (c->eos != OX_EOS_IDEAL && c->eos != OX_EOS_GAS_RADIATION) return OX_ERR_UNSUPPORTED;
  if (c->eos == OX_EOS_GAS_RADIATION && (!(c->eos_R > 0.0) || !(c->eos_ar > 0.0))) return OX_ERR_INVALID_ARG;
  if (!(c->gamma > 1.0)) return OX_ERR_INVALID_ARG;
  if (c->riemann != OX_RIEMANN_HLL && c->riemann != OX_RIEMANN_HLLC) return OX_ERR_INVALID_ARG;
  if (c->limiter < OX_LIM_NONE || c->limiter > OX_LIM_MC) return OX_ERR_INVALID_ARG;
  if (c->n_scalars < 0 || 2 + c->ndim + c->n_scalars > NVMAX) return OX_ERR_INVALID_ARG;
  if (c->gravity < OX_GRAV_NONE || c->gravity > OX_GRAV_SELF) return OX_ERR_INVALID_ARG;
  if ((c->gravity == OX_GRAV_POINT_MASS || c->gravity == OX_GRAV_SELF) && c->coords != OX_SPHERICAL) return OX_ERR_INVALID_ARG;
  for (int d = 0; d < 3; ++d) {
    if (d < c->ndim) {
      if (c->n[d] < NG) return OX_ERR_INVALID_ARG;
      if (c->bc_lo[d] < 0 || c->bc_lo[d] > OX_BC_WEDGE || c->bc_hi[d] < 0 || c->bc_hi[d] > OX_BC_WEDGE)
        return OX_ERR_INVALID_ARG;
      if ((c->bc_lo[d] == OX_BC_PERIODIC) != (c->bc_hi[d] == OX_BC_PERIODIC)) return OX_ERR_INVALID_ARG;
      if (c->coords == OX_SPHERICAL && d == 0 && c->bc_lo[d] == OX_BC_PERIODIC) return OX_ERR_INVALID_ARG;
      if (c->spacing[d] == OX_SPACING_CUSTOM) {
        if (!c->faces[d]) return OX_ERR_INVALID_ARG;
        for (int i = 0; i < c->n[d]; ++i)
          if (!(c->faces[d][i + 1] > c->faces[d][i])) return OX_ERR_INVALID_ARG;
      } else {
        if (!(c->hi[d] > c->lo[d])) return OX_ERR_INVALID_ARG;
        if (c->spacing[d] == OX_SPACING_LOG && !(c->lo[d] > 0.0)) return OX_ERR_INVALID_ARG;
        if (c->spacing[d] != OX_SPACING_UNIFORM && c->spacing[d] != OX_SPACING_LOG) return OX_ERR_INVALID_ARG;
      }
    } else if (c->n[d] != 1) {
      return OX_ERR_INVALID_ARG;
    }
  }
  return OX_OK;
}

}  // namespace

extern "C" {

int ox_create(const ox_config* cfg, ox_handle** out) {
  if (!out) return OX_ERR_INVALID_ARG;
  *out = nullptr;
  const int rc = check_config(cfg);
  if (rc != OX_OK) return rc;
  ox_handle* h = new (std::nothrow) ox_handle();
  if (!h) return OX_ERR_ALLOC;
  h->c = *cfg;
  h->nvar = 2 + cfg->ndim + cfg->n_scalars;
  const double PI = 3.14159265358979323846;
  for (int d = 0; d < 3; ++d) {
    const bool active = d < cfg->ndim;
    const int n = cfg->n[d];
    h->ng[d] = active ? NG : 0;
    h->np[d] = n + 2 * h->ng[d];
    std::vector<double>& xf = h->xf[d];
    xf.assign(h->np[d] + 1, 0.0);
    double* f = xf.data() + h->ng[d];  // f[i] = minus face of interior cell i, i = 0..n
    if (!active) {
      double lo = cfg->lo[d], hi = cfg->hi[d];
      if (!(hi > lo)) {
        lo = 0.0;
        hi = 1.0;
        if (cfg->coords == OX_SPHERICAL) hi = (d == 1) ? PI : 2.0 * PI;
      }
      f[0] = lo;
      f[1] = hi;
      continue;
    }
    if (cfg->spacing[d] == OX_SPACING_CUSTOM) {
      for (int i = 0; i <= n; ++i) f[i] = cfg->faces[d][i];
    } else if (cfg->spacing[d] == OX_SPACING_LOG) {
      for (int i = 0; i <= n; ++i) f[i] = cfg->lo[d] * std::pow(cfg->hi[d] / cfg->lo[d], (double)i / (double)n);
      f[0] = cfg->lo[d];
      f[n] = cfg->hi[d];
    } else {
      for (int i = 0; i <= n; ++i) f[i] = cfg->lo[d] + (double)i * (cfg->hi[d] - cfg->lo[d]) / (double)n;
      f[n] = cfg->hi[d];
    }
    // ghost geometry: widths copied from the far side (periodic) or mirrored about the boundary
    for (int g = 1; g <= NG; ++g) {
      const double wlo = (cfg->bc_lo[d] == OX_BC_PERIODIC) ? (f[n - g + 1] - f[n - g]) : (f[g] - f[g - 1]);
      f[-g] = f[-g + 1] - wlo;
      const double whi = (cfg->bc_hi[d] == OX_BC_PERIODIC) ? (f[g] - f[g - 1]) : (f[n - g + 1] - f[n - g]);
      f[n + g] = f[n + g - 1] + whi;
    }
  }
  h->ncp = (size_t)h->np[0] * h->np[1] * h->np[2];
  try {
    h->U.assign((size_t)h->nvar * h->ncp, 0.0);
  } catch (...) {
    delete h;
    return OX_ERR_ALLOC;
  }
  h->c.faces[0] = h->c.faces[1] = h->c.faces[2] = nullptr;  // caller's arrays are not retained
  *out = h;
  return OX_OK;
}

int ox_destroy(ox_handle* h) {
  delete h;
  return OX_OK;
}

int ox_nvar(const ox_handle* h) { return h ? h->nvar : OX_ERR_INVALID_ARG; }

int ox_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

int ox_set_state(ox_handle* h, const double* data, int form) {
  if (!h || !data || (form != OX_CONSERVED && form != OX_PRIMITIVE)) return OX_ERR_INVALID_ARG;
  h->gself_dirty = true;
  const ox_config& c = h->c;
  const size_t nint = (size_t)c.n[0] * c.n[1] * c.n[2];
#pragma omp parallel for if (h->ncp > 32768)
  for (int k = 0; k < c.n[2]; ++k)
    for (int j = 0; j < c.n[1]; ++j)
      for (int i = 0; i < c.n[0]; ++i) {
        const size_t src = ((size_t)k * c.n[1] + j) * c.n[0] + i;
        double a[NVMAX], b[NVMAX];
        for (int v = 0; v < h->nvar; ++v) a[v] = data[(size_t)v * nint + src];
        if (form == OX_PRIMITIVE) {
          prim_to_cons(eos_of(c), c.ndim, h->nvar, a, b);
        } else {
          for (int v = 0; v < h->nvar; ++v) b[v] = a[v];
        }
        const size_t dst = h->cell(i, j, k);
        for (int v = 0; v < h->nvar; ++v) h->U[(size_t)v * h->ncp + dst] = b[v];
      }
  return OX_OK;
}

int ox_get_state(ox_handle* h, double* data, int form) {
  if (!h || !data || (form != OX_CONSERVED && form != OX_PRIMITIVE)) return OX_ERR_INVALID_ARG;
  const ox_config& c = h->c;
  const size_t nint = (size_t)c.n[0] * c.n[1] * c.n[2];
#pragma omp parallel for if (h->ncp > 32768)
  for (int k = 0; k < c.n[2]; ++k)
    for (int j = 0; j < c.n[1]; ++j)
      for (int i = 0; i < c.n[0]; ++i) {
        const size_t dst = ((size_t)k * c.n[1] + j) * c.n[0] + i;
        const size_t src = h->cell(i, j, k);
        double a[NVMAX], b[NVMAX];
        for (int v = 0; v < h->nvar; ++v) a[v] = h->U[(size_t)v * h->ncp + src];
        if (form == OX_PRIMITIVE) {
          cons_to_prim(eos_of(c), c.ndim, h->nvar, a, b);
        } else {
          for (int v = 0; v < h->nvar; ++v) b[v] = a[v];
        }
        for (int v = 0; v < h->nvar; ++v) data[(size_t)v * nint + dst] = b[v];
      }
  return OX_OK;
}

// O7 (reading R2): rate_i = sum over active d of (|u_d| + c_s)/l_d with l = (dr, r_c dtheta,
// r_c sin(theta_c) dphi) in spherical coordinates, cell widths in Cartesian; dt = cfl / max rate.
int ox_compute_dt(ox_handle* h, double cfl, double* dt_out) {
  if (!h || !dt_out || !(cfl > 0.0)) return OX_ERR_INVALID_ARG;
  const ox_config& c = h->c;
  double rmax = 0.0;
  int bad = 0;
#pragma omp parallel for reduction(max : rmax) reduction(| : bad) if (h->ncp > 32768)
  for (int k = 0; k < c.n[2]; ++k)
    for (int j = 0; j < c.n[1]; ++j)
      for (int i = 0; i < c.n[0]; ++i) {
        const size_t ci = h->cell(i, j, k);
        double U[NVMAX], W[NVMAX];
        for (int v = 0; v < h->nvar; ++v) U[v] = h->U[(size_t)v * h->ncp + ci];
        cons_to_prim(eos_of(c), c.ndim, h->nvar, U, W);
        const double rho = W[0], P = W[1 + c.ndim];
        if (!(rho > 0.0) || !(P > 0.0) || !std::isfinite(rho) || !std::isfinite(P)) {
          bad = 1;
          continue;
        }
        const double cs = eos_sound_speed(eos_of(c), rho, P);
        const int id[3] = {i, j, k};
        double rate = 0.0;
        for (int d = 0; d < c.ndim; ++d) {
          double len = h->width(d, id[d]);
          if (c.coords == OX_SPHERICAL) {
            if (d == 1) len *= h->xc(0, i);
            if (d == 2) len *= h->xc(0, i) * std::sin(h->xc(1, j));
          }
          rate += (std::fabs(W[1 + d]) + cs) / len;
        }
        if (!std::isfinite(rate)) bad = 1;
        rmax = std::max(rmax, rate);
      }
  if (bad) return OX_ERR_NONPHYSICAL;
  *dt_out = cfl / rmax;
  return OX_OK;
}

int ox_step(ox_handle* h, double dt) {
  if (!h || !(dt > 0.0)) return OX_ERR_INVALID_ARG;
  const ox_config& c = h->c;
  const int ndim = c.ndim, nvar = h->nvar;
  const size_t ncp = h->ncp;
  std::vector<double>& U = h->U;

  refresh_self_gravity(h);   // Eq. 4 from U^n (reading R28)
  fill_ghosts(h, U);  // O0

  std::vector<double> W((size_t)nvar * ncp);  // O1 on every padded cell
#pragma omp parallel for if (h->ncp > 32768)
  for (long long ci = 0; ci < (long long)ncp; ++ci) {
    double a[NVMAX], b[NVMAX];
    for (int v = 0; v < nvar; ++v) a[v] = U[(size_t)v * ncp + ci];
    cons_to_prim(eos_of(c), ndim, nvar, a, b);
    for (int v = 0; v < nvar; ++v) W[(size_t)v * ncp + ci] = b[v];
  }

  // O2-O4: predicted face states on interior + one ring
  std::vector<double> Um[3], Up[3];
  for (int d = 0; d < ndim; ++d) {
    Um[d].assign((size_t)nvar * ncp, 0.0);
    Up[d].assign((size_t)nvar * ncp, 0.0);
  }
  std::vector<double> Pbar(ncp, 0.0);
  int lo[3], hi[3];
  for (int d = 0; d < 3; ++d) {
    lo[d] = (d < ndim) ? -1 : 0;
    hi[d] = (d < ndim) ? c.n[d] + 1 : 1;
  }
#pragma omp parallel for if (h->ncp > 32768)
  for (int k = lo[2]; k < hi[2]; ++k)
    for (int j = lo[1]; j < hi[1]; ++j)
      for (int i = lo[0]; i < hi[0]; ++i) {
        const size_t ci = h->cell(i, j, k);
        double Wc[NVMAX], Wn[3][2][NVMAX];
        for (int v = 0; v < nvar; ++v) Wc[v] = W[(size_t)v * ncp + ci];
        for (int d = 0; d < ndim; ++d) {
          int a[3] = {i, j, k}, b[3] = {i, j, k};
          a[d] -= 1;
          b[d] += 1;
          const size_t ca = h->cell(a[0], a[1], a[2]), cb = h->cell(b[0], b[1], b[2]);
          for (int v = 0; v < nvar; ++v) {
            Wn[d][0][v] = W[(size_t)v * ncp + ca];
            Wn[d][1][v] = W[(size_t)v * ncp + cb];
          }
        }
        double um[3][NVMAX], up[3][NVMAX], pb;
        predictor(h, i, j, k, dt, Wc, Wn, um, up, pb);
        for (int d = 0; d < ndim; ++d)
          for (int v = 0; v < nvar; ++v) {
            Um[d][(size_t)v * ncp + ci] = um[d][v];
            Up[d][(size_t)v * ncp + ci] = up[d][v];
          }
        Pbar[ci] = pb;
      }

  // O5: F[d] at cell ci = Riemann flux through the MINUS face of that cell in direction d
  std::vector<double> F[3];
  for (int d = 0; d < ndim; ++d) {
    F[d].assign((size_t)(nvar + 2) * ncp, 0.0);   // + advective flux of e and face velocity (monitoring)
    int fhi[3] = {c.n[0], c.n[1], c.n[2]};
    fhi[d] += 1;
#pragma omp parallel for if (h->ncp > 32768)
    for (int k = 0; k < fhi[2]; ++k)
      for (int j = 0; j < fhi[1]; ++j)
        for (int i = 0; i < fhi[0]; ++i) {
          int a[3] = {i, j, k};
          a[d] -= 1;
          const size_t cl = h->cell(a[0], a[1], a[2]), cr = h->cell(i, j, k);
          double UL[NVMAX], UR[NVMAX], Fl[NFMAX];
          for (int v = 0; v < nvar; ++v) {
            UL[v] = Up[d][(size_t)v * ncp + cl];
            UR[v] = Um[d][(size_t)v * ncp + cr];
          }
          riemann_flux(c.riemann, eos_of(c), ndim, nvar, d, UL, UR, Fl);
          for (int v = 0; v < nvar + 2; ++v) F[d][(size_t)v * ncp + cr] = Fl[v];
        }
  }

  // O6
  std::vector<double> Unew(U);
#pragma omp parallel for if (h->ncp > 32768)
  for (int k = 0; k < c.n[2]; ++k)
    for (int j = 0; j < c.n[1]; ++j)
      for (int i = 0; i < c.n[0]; ++i) {
        const size_t ci = h->cell(i, j, k);
        double Un[NVMAX], Fm[3][NFMAX], Fp[3][NFMAX], out[NVMAX];
        for (int v = 0; v < nvar; ++v) Un[v] = U[(size_t)v * ncp + ci];
        for (int d = 0; d < ndim; ++d) {
          int b[3] = {i, j, k};
          b[d] += 1;
          const size_t cp = h->cell(b[0], b[1], b[2]);
          for (int v = 0; v < nvar + 2; ++v) {
            Fm[d][v] = F[d][(size_t)v * ncp + ci];
            Fp[d][v] = F[d][(size_t)v * ncp + cp];
          }
        }
        const double* fm[3] = {Fm[0], Fm[1], Fm[2]};
        const double* fp[3] = {Fp[0], Fp[1], Fp[2]};
        update_cell(h, i, j, k, dt, Un, fm, fp, Pbar[ci], out);
        for (int v = 0; v < nvar; ++v) Unew[(size_t)v * ncp + ci] = out[v];
      }
  U.swap(Unew);
  h->gself_dirty = true;
  return OX_OK;
}

int ox_cell_update(ox_handle* h, int i, int j, int k, double dt, double* out) {
  if (!h || !out || !(dt > 0.0)) return OX_ERR_INVALID_ARG;
  const ox_config& c = h->c;
  if (i < 0 || i >= c.n[0] || j < 0 || j >= c.n[1] || k < 0 || k >= c.n[2]) return OX_ERR_INVALID_ARG;
  refresh_self_gravity(h);
  double Un[NVMAX], Fm[3][NFMAX], Fp[3][NFMAX];
  naive_get_U(h, i, j, k, Un);
  for (int d = 0; d < c.ndim; ++d) {
    int b[3] = {i, j, k};
    b[d] += 1;
    naive_face_flux(h, i, j, k, d, dt, Fm[d]);
    naive_face_flux(h, b[0], b[1], b[2], d, dt, Fp[d]);
  }
  double um[3][NVMAX], up[3][NVMAX], pbar;
  naive_predict(h, i, j, k, dt, um, up, pbar);
  const double* fm[3] = {Fm[0], Fm[1], Fm[2]};
  const double* fp[3] = {Fp[0], Fp[1], Fp[2]};
  update_cell(h, i, j, k, dt, Un, fm, fp, pbar, out);
  return OX_OK;
}

int ox_riemann_flux(int riemann, double gamma, int ndim, int ns, int dir, const double* UL, const double* UR,
                    double* F) {
  if (ndim < 1 || ndim > 3 || ns < 0 || 2 + ndim + ns > NVMAX || dir < 0 || dir >= ndim) return OX_ERR_INVALID_ARG;
  riemann_flux_core(riemann, gamma, ndim, 2 + ndim + ns, dir, UL, UR, F);
  return OX_OK;
}

int ox_physical_flux(double gamma, int ndim, int ns, int dir, const double* U, double* F) {
  if (ndim < 1 || ndim > 3 || ns < 0 || 2 + ndim + ns > NVMAX || dir < 0 || dir >= ndim) return OX_ERR_INVALID_ARG;
  double W[NVMAX];
  cons_to_prim(gamma, ndim, 2 + ndim + ns, U, W);
  flux_from_prim(gamma, ndim, 2 + ndim + ns, dir, W, F);
  return OX_OK;
}


int ox_self_gravity(ox_handle* h, int i, double* g_out) {
  if (!h || !g_out || h->c.gravity != OX_GRAV_SELF || i < 0 || i >= h->c.n[0]) return OX_ERR_INVALID_ARG;
  refresh_self_gravity(h);
  *g_out = h->gself[i];
  return OX_OK;
}

double ox_eos_pressure(int eos, double gamma, double R, double ar, double rho, double e) { return eos_pressure(Eos(eos, gamma, R, ar), rho, e); }
double ox_eos_energy(int eos, double gamma, double R, double ar, double rho, double P) { return eos_energy(Eos(eos, gamma, R, ar), rho, P); }
double ox_eos_sound_speed(int eos, double gamma, double R, double ar, double rho, double P) {
  return eos_sound_speed(Eos(eos, gamma, R, ar), rho, P);
}

double ox_limiter(int lim, double a, double b) { return limiter(lim, a, b); }

int ox_cell_geometry(const ox_handle* h, int i, int j, int k, double* dV, double* dS6, double* xc3) {
  if (!h) return OX_ERR_INVALID_ARG;
  const int id[3] = {i, j, k};
  for (int d = 0; d < 3; ++d)
    if (id[d] < -h->ng[d] || id[d] >= h->c.n[d] + h->ng[d]) return OX_ERR_INVALID_ARG;
  double v, s[3][2];
  cell_geometry(h, i, j, k, v, s);
  if (dV) *dV = v;
  if (dS6)
    for (int d = 0; d < 3; ++d) {
      dS6[2 * d] = s[d][0];
      dS6[2 * d + 1] = s[d][1];
    }
  if (xc3)
    for (int d = 0; d < 3; ++d) xc3[d] = h->xc(d, id[d]);
  return OX_OK;
}

int ox_faces(const ox_handle* h, int d, double* out) {
  if (!h || !out || d < 0 || d > 2) return OX_ERR_INVALID_ARG;
  std::memcpy(out, h->xf[d].data(), h->xf[d].size() * sizeof(double));
  return OX_OK;
}

}  // extern "C"

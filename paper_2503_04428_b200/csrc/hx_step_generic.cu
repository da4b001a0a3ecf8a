// hx_step_generic.cu -- straightforward one-thread-per-cell version of the unsplit MUSCL-Hancock
// step (A1-A7 of SURVEY 8(a)) for any ndim / geometry / nvar.  Reads the ghost-filled padded
// state from global memory (L1/L2 serve the 13-point-star re-reads) and recomputes the
// neighbours' predictors redundantly.  It is the correctness-first path, the path for shapes
// the fused tile kernel does not cover, and the on-device cross-check of the tile kernel.
//
// PAPER.md: Eq. 17 (slopes, face states), Eq. 18 (half-step predictor, unsplit per Toro 16.5),
// Eq. 19 (Godunov update), Eq. 13-16 (spherical sources), Eq. 2-3 (gravity).
#include "hx_common.cuh"

namespace hx {

template <int ND, bool SPH>
__device__ __forceinline__ void face_coeffs(const Tables& T, int pi, int pj, int pk, double cm[ND], double cp[ND]) {
#pragma unroll
  for (int d = 0; d < ND; ++d) {
    if (!SPH) {
      const int p = (d == 0) ? pi : (d == 1 ? pj : pk);
      cm[d] = cp[d] = T.cf[d][0][d][p];
    } else {
      cm[d] = T.cf[d][0][0][pi] * T.cf[d][0][1][pj] * T.cf[d][0][2][pk];
      cp[d] = T.cf[d][1][0][pi] * T.cf[d][1][1][pj] * T.cf[d][1][2][pk];
    }
  }
}

template <int ND, int NVA>
__device__ __forceinline__ void load_prim(const StepArgs& a, int nv, long long o, double* W) {
  double U[NVA];
  for (int v = 0; v < nv; ++v) U[v] = __ldg(a.Uin + v * a.L.sv + o);
  cons_to_prim<ND>(a.P, nv, U, W);
}

// O1-O4 for the cell at padded index (pi,pj,pk): primitives W, limited slopes sig[d], half-step
// increment dU (conserved), and the pressure of the cell-centred predicted state.
template <int ND, bool SPH, int NVA>
__device__ __noinline__ void predict_cell(const StepArgs& a, int nv, int pi, int pj, int pk, double* W, double (*sig)[NVA],
                                          double* dU, double* pbar) {
  const Layout& L = a.L;
  const long long o = L.off(pi, pj, pk);
  load_prim<ND, NVA>(a, nv, o, W);
  for (int v = 0; v < nv; ++v) dU[v] = 0.0;
  if (a.P.limiter == HX_LIM_NONE) {   // R19: first-order Godunov
#pragma unroll
    for (int d = 0; d < ND; ++d)
      for (int v = 0; v < nv; ++v) sig[d][v] = 0.0;
    *pbar = W[1 + ND];
    return;
  }
  double cm[ND], cp[ND];
  face_coeffs<ND, SPH>(a.T, pi, pj, pk, cm, cp);
  const int pidx[3] = {pi, pj, pk};
  const long long strides[3] = {1, L.sy, L.sz};
  double U[NVA];
  prim_to_cons<ND>(a.P, nv, W, U);
#pragma unroll
  for (int d = 0; d < ND; ++d) {
    double Wm[NVA], Wp[NVA];
    load_prim<ND, NVA>(a, nv, o - strides[d], Wm);
    load_prim<ND, NVA>(a, nv, o + strides[d], Wp);
    const int p = pidx[d];
    const double ia = a.T.idx[d][p], ib = a.T.idx[d][p + 1], hw = a.T.hw[d][p];
    double Wf[NVA], Uf[NVA], Ff[NVA];
    for (int v = 0; v < nv; ++v) sig[d][v] = limited_slope(a.P.limiter, (W[v] - Wm[v]) * ia, (Wp[v] - W[v]) * ib);
    for (int v = 0; v < nv; ++v) Wf[v] = W[v] - hw * sig[d][v];
    prim_to_cons<ND>(a.P, nv, Wf, Uf);
    flux_along<ND>(nv, d, Wf, Uf, Ff);
    for (int v = 0; v < nv; ++v) dU[v] += Ff[v] * cm[d];
    for (int v = 0; v < nv; ++v) Wf[v] = W[v] + hw * sig[d][v];
    prim_to_cons<ND>(a.P, nv, Wf, Uf);
    flux_along<ND>(nv, d, Wf, Uf, Ff);
    for (int v = 0; v < nv; ++v) dU[v] -= Ff[v] * cp[d];
  }
  if (SPH) {   // cell-centred geometric sources (R8)
    const double rho = W[0], ur = W[1], ut = (ND >= 2) ? W[2] : 0.0, up = (ND >= 3) ? W[3] : 0.0, p = W[1 + ND];
    dU[1] += (rho * ut * ut + rho * up * up + 2.0 * p) * a.T.gr[pi];
    if (ND >= 2) dU[2] += -rho * ut * ur * a.T.Ar[pi] + (rho * up * up + p) * a.T.cr[pi] * a.T.gt[pj];
    if (ND >= 3) dU[3] += -rho * up * ur * a.T.Ar[pi] - rho * up * ut * a.T.cr[pi] * a.T.At[pj];
  }
  if (a.P.gravity != HX_GRAV_NONE) {
#pragma unroll
    for (int d = 0; d < ND; ++d) {
      const double g = a.T.grav[d][pidx[d]];
      dU[1 + d] += W[0] * g;
      dU[1 + ND] += U[1 + d] * g;
    }
  }
  const double hdt = 0.5 * a.dt;
  for (int v = 0; v < nv; ++v) dU[v] *= hdt;
  double Uc[NVA], Wc[NVA];
  for (int v = 0; v < nv; ++v) Uc[v] = U[v] + dU[v];
  cons_to_prim<ND>(a.P, nv, Uc, Wc);
  *pbar = Wc[1 + ND];
}

// Predicted conservative state on the minus (side = -1) or plus (+1) face of direction d.
template <int ND, int NVA>
__device__ __forceinline__ void face_state(const Phys& P, int nv, const double* W, const double* sig, double hw, double side,
                                           const double* dU, double* Uf) {
  double Wf[NVA];
  for (int v = 0; v < nv; ++v) Wf[v] = W[v] + side * hw * sig[v];
  prim_to_cons<ND>(P, nv, Wf, Uf);
  for (int v = 0; v < nv; ++v) Uf[v] += dU[v];
}

template <int ND, bool SPH, int NVC>
__global__ void __launch_bounds__(128) step_generic_kernel(StepArgs a) {
  constexpr int NVA = NVC ? NVC : NVMAX;
  const Layout& L = a.L;
  const int nv = NVC ? NVC : L.nvar;
  const long long ncell = (long long)L.n[0] * L.n[1] * L.n[2];
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  double rate = 0.0;
  if (tid < ncell) {
    const int i = (int)(tid % L.n[0]);
    const int j = (int)((tid / L.n[0]) % L.n[1]);
    const int k = (int)(tid / ((long long)L.n[0] * L.n[1]));
    const int pidx[3] = {i + L.ng[0], j + L.ng[1], k + L.ng[2]};
    const long long o = L.off(pidx[0], pidx[1], pidx[2]);

    double Wc[NVA], sigc[ND][NVA], dUc[NVA], pbar;
    predict_cell<ND, SPH, NVA>(a, nv, pidx[0], pidx[1], pidx[2], Wc, sigc, dUc, &pbar);
    double cm[ND], cp[ND];
    face_coeffs<ND, SPH>(a.T, pidx[0], pidx[1], pidx[2], cm, cp);

    double acc[NVA];
    for (int v = 0; v < nv; ++v) acc[v] = 0.0;
    double FmM[ND][ND], FpM[ND][ND];   // momentum components of the face fluxes (spherical sources)
    const bool emon = a.P.emon_eps > 0.0;
    double eadv = 0.0, divu = 0.0;      // Eq. 10 in finite-volume form: -div(u e) and div u from the face quantities
#pragma unroll
    for (int d = 0; d < ND; ++d) {
      int q[3] = {pidx[0], pidx[1], pidx[2]};
      double Wn[NVA], sign[ND][NVA], dUn[NVA], pb, UL[NVA], UR[NVA], F[NVA];
      const double hwc = a.T.hw[d][pidx[d]];
      // minus face: neighbour's plus state | own minus state
      q[d] = pidx[d] - 1;
      predict_cell<ND, SPH, NVA>(a, nv, q[0], q[1], q[2], Wn, sign, dUn, &pb);
      face_state<ND, NVA>(a.P, nv, Wn, sign[d], a.T.hw[d][q[d]], 1.0, dUn, UL);
      face_state<ND, NVA>(a.P, nv, Wc, sigc[d], hwc, -1.0, dUc, UR);
      riemann_flux<ND, NVA>(a.P, nv, d, UL, UR, F);
      for (int v = 0; v < nv; ++v) acc[v] += F[v] * cm[d];
      if (emon) {
        double phi, uf;
        monitor_face<ND, NVA>(a.P, nv, d, UL, UR, F[0], phi, uf);
        eadv += phi * cm[d];
        divu -= uf * cm[d];
      }
#pragma unroll
      for (int e = 0; e < ND; ++e) FmM[d][e] = F[1 + e];
      // plus face: own plus state | neighbour's minus state
      q[d] = pidx[d] + 1;
      predict_cell<ND, SPH, NVA>(a, nv, q[0], q[1], q[2], Wn, sign, dUn, &pb);
      face_state<ND, NVA>(a.P, nv, Wc, sigc[d], hwc, 1.0, dUc, UL);
      face_state<ND, NVA>(a.P, nv, Wn, sign[d], a.T.hw[d][q[d]], -1.0, dUn, UR);
      riemann_flux<ND, NVA>(a.P, nv, d, UL, UR, F);
      for (int v = 0; v < nv; ++v) acc[v] -= F[v] * cp[d];
      if (emon) {
        double phi, uf;
        monitor_face<ND, NVA>(a.P, nv, d, UL, UR, F[0], phi, uf);
        eadv -= phi * cp[d];
        divu += uf * cp[d];
      }
#pragma unroll
      for (int e = 0; e < ND; ++e) FpM[d][e] = F[1 + e];
    }

    double Un[NVA], Unew[NVA];
    for (int v = 0; v < nv; ++v) Un[v] = __ldg(a.Uin + v * L.sv + o);
    for (int v = 0; v < nv; ++v) Unew[v] = Un[v] + a.dt * acc[v];
    if (SPH) {   // Eq. 14-16 from the face Riemann fluxes (R9-R11); Pbar stands in for inactive angular faces
      const int pi = pidx[0], pj = pidx[1];
      const double Ftt = (ND >= 2) ? 0.5 * (FmM[ND >= 2 ? 1 : 0][ND >= 2 ? 1 : 0] + FpM[ND >= 2 ? 1 : 0][ND >= 2 ? 1 : 0]) : pbar;
      const double Fpp = (ND >= 3) ? 0.5 * (FmM[ND >= 3 ? 2 : 0][ND >= 3 ? 2 : 0] + FpM[ND >= 3 ? 2 : 0][ND >= 3 ? 2 : 0]) : pbar;
      Unew[1] += a.dt * ((Ftt + Fpp) * a.T.gr[pi]);
      if (ND >= 2) {
        const int t = ND >= 2 ? 1 : 0;
        Unew[2] += a.dt * (-a.T.rr[pi] * (FpM[0][t] * cp[0] + FmM[0][t] * cm[0]) + Fpp * a.T.cr[pi] * a.T.gt[pj]);
      }
      if (ND >= 3) {
        const int t = ND >= 3 ? 1 : 0, f = ND >= 3 ? 2 : 0;
        Unew[3] += a.dt * (-a.T.rr[pi] * (FpM[0][f] * cp[0] + FmM[0][f] * cm[0]) -
                           a.T.st[pj] * (FpM[t][f] * cp[t] + FmM[t][f] * cm[t]));
      }
    }
    if (a.P.gravity != HX_GRAV_NONE) {   // time-centred (R13)
#pragma unroll
      for (int d = 0; d < ND; ++d) {
        const double g = a.T.grav[d][pidx[d]];
        const double mnew = Unew[1 + d] + a.dt * 0.5 * (Un[0] + Unew[0]) * g;
        Unew[1 + ND] += a.dt * 0.5 * (Un[1 + d] + mnew) * g;
        Unew[1 + d] = mnew;
      }
    }
    if (emon) {   // Eq. 11-12: e^{n+1} from the blend, E reset to e_k + e (R29)
      double kn = 0.0, k1 = 0.0;
#pragma unroll
      for (int d = 0; d < ND; ++d) {
        kn += Un[1 + d] * Un[1 + d];
        k1 += Unew[1 + d] * Unew[1 + d];
      }
      const double en = Un[1 + ND] - 0.5 * kn / Un[0], ek = 0.5 * k1 / Unew[0];
      const double e1 = Unew[1 + ND] - ek;
      const double e2 = en + a.dt * (eadv - Wc[1 + ND] * divu);
      Unew[1 + ND] = ek + monitor_blend(a.P.emon_eps, en, e1, e2, ek);
    }
    for (int v = 0; v < nv; ++v) a.Uout[v * L.sv + o] = Unew[v];

    // A7 folded in: CFL rate of the new state + positivity check
    double Wn[NVA];
    cons_to_prim<ND>(a.P, nv, Unew, Wn);
    const double rho = Wn[0], p = Wn[1 + ND];
    if (!(rho > 0.0) || !(p > 0.0) || !isfinite(rho) || !isfinite(p)) {
      atomicOr(a.status, 1);
    } else {
      const double cs = eos_sound_speed(a.P, rho, p);
#pragma unroll
      for (int d = 0; d < ND; ++d) {
        const double il = a.T.lf[d][0][pidx[0]] * a.T.lf[d][1][pidx[1]] * a.T.lf[d][2][pidx[2]];
        rate += (fabs(Wn[1 + d]) + cs) * il;
      }
      if (!isfinite(rate)) {
        atomicOr(a.status, 1);
        rate = 0.0;
      }
    }
  }
  block_rate_max(rate, a.rate_bits);
}

template <int ND, bool SPH>
static cudaError_t launch_nd(const StepArgs& a, cudaStream_t s) {
  const long long ncell = (long long)a.L.n[0] * a.L.n[1] * a.L.n[2];
  const unsigned grid = (unsigned)((ncell + 127) / 128);
  switch (a.L.nvar - ND - 2) {   // number of passive scalars: common counts get register-resident arrays
    case 0: step_generic_kernel<ND, SPH, ND + 2><<<grid, 128, 0, s>>>(a); break;
    case 1: step_generic_kernel<ND, SPH, ND + 3><<<grid, 128, 0, s>>>(a); break;
    case 2: step_generic_kernel<ND, SPH, ND + 4><<<grid, 128, 0, s>>>(a); break;
    case 4: step_generic_kernel<ND, SPH, ND + 6><<<grid, 128, 0, s>>>(a); break;
    default: step_generic_kernel<ND, SPH, 0><<<grid, 128, 0, s>>>(a); break;
  }
  return cudaGetLastError();
}

cudaError_t launch_step_generic(const StepArgs& a, cudaStream_t s) {
  const bool sph = a.P.spherical != 0;
  switch (a.L.ndim) {
    case 1: return sph ? launch_nd<1, true>(a, s) : launch_nd<1, false>(a, s);
    case 2: return sph ? launch_nd<2, true>(a, s) : launch_nd<2, false>(a, s);
    default: return sph ? launch_nd<3, true>(a, s) : launch_nd<3, false>(a, s);
  }
}

}  // namespace hx

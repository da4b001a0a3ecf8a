// hx_host.cu -- the C ABI of include/hx.h: configuration checks, padded state allocation, 1-D
// geometry tables (PAPER.md: dS and dV "computed based on the chosen geometry"), and the
// per-step launch sequence  ghost fill -> fused step (+ CFL rate)  on the handle's stream.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "hx_common.cuh"

namespace hx {
cudaError_t launch_ghost_fill(const Layout& L, double* U, const int* bc_lo, const int* bc_hi, int skip_x, cudaStream_t s);
cudaError_t launch_pack(const Layout& L, const Phys& P, const double* src, double* U, int to_cons, cudaStream_t s);
cudaError_t launch_unpack(const Layout& L, const Phys& P, const double* U, double* dst, int to_prim, cudaStream_t s);
cudaError_t launch_rate(const Layout& L, const Tables& T, const Phys& P, const double* U, unsigned long long* rate_bits, int* status,
                        cudaStream_t s);
cudaError_t launch_step_generic(const StepArgs& a, cudaStream_t s);
cudaError_t launch_self_gravity(const Layout& L, const double* U, const double* const xf[3], double* partial, int groups, double* grav_r,
                                double GM, double G, int bc_lo, int bc_hi, double* weights, bool* weights_ready, cudaStream_t s);
namespace t2 { struct Plan; }
int tile2_supported(const Layout& L, const Phys& P);
cudaError_t tile2_plan_create(const Layout& L, const Phys& P, double* const U[2], const double* uni, int grav_z, int bcx_lo, int bcx_hi, t2::Plan** out);
int tile2_writes_x_ghosts(const t2::Plan* p);
void tile2_plan_destroy(t2::Plan* p);
cudaError_t launch_step_tile2(t2::Plan* plan, const StepArgs& a, int cur, cudaStream_t s);
const char* tile2_kernel_name(const t2::Plan* p);
}  // namespace hx

using namespace hx;

struct DevScalars {   // device-resident scalars read back by hx_compute_dt in one copy
  unsigned long long rate_bits;
  int status;
  int pad;
};

struct hx_handle {
  hx_config cfg;
  Layout L;
  Tables T;
  Phys P;
  double* d_U[2] = {nullptr, nullptr};
  int cur = 0;
  double* d_tables = nullptr;
  DevScalars* d_scal = nullptr;
  DevScalars* h_scal = nullptr;   // pinned
  cudaStream_t stream = nullptr;
  cudaStream_t side = nullptr;    // reads the CFL rate back while the next ghost fill already runs on `stream`
  cudaEvent_t ev_step = nullptr;  // recorded right after the step kernel
  const double* d_xf[3] = {nullptr, nullptr, nullptr};   // padded face coordinates on the device (self-gravity)
  double* d_grav_r = nullptr;     // the radial acceleration table inside d_tables (rewritten every step by self-gravity)
  double* d_sg_partial = nullptr; // self-gravity: partial shell sums [sg_groups][n0], then the angular weights [n1 + n2]
  bool sg_weights_ready = false;
  int sg_groups = 0;
  bool ghosts_valid = false;      // ghost layers of d_U[cur] are filled (hx_step fills them eagerly for the next step)
  bool rate_valid = false;
  int kernel_opt = HX_KERNEL_AUTO;
  t2::Plan* plan2 = nullptr;
  bool plan2_tried = false;
  bool uniform = false;       // Cartesian grid whose per-axis tables are bitwise constant
  double uni[6] = {0, 0, 0, 0, 0, 0};   // hw*idx and 1/delta of the three axes when uniform
  long long launches = 0;
  const char* last_kernel = "none";
  bool async_host = false;    // HX_OPT_ASYNC_HOST: host-buffer copies are only enqueued
  bool timing = false, ev_pending = false;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  double kernel_ms = 0.0;
  long long kernel_launches = 0;
  char err[256] = {0};
};

namespace {

int fail(hx_handle* h, int code, const char* fmt, const char* detail = "") {
  if (h) snprintf(h->err, sizeof(h->err), fmt, detail);
  return code;
}

int cuda_fail(hx_handle* h, cudaError_t e, const char* where) {
  if (h) snprintf(h->err, sizeof(h->err), "%s: %s", where, cudaGetErrorString(e));
  return HX_ERR_CUDA;
}

bool reflecting(int bc) { return bc == HX_BC_REFLECTING || bc == HX_BC_WEDGE; }

const char* check_config(const hx_config* c, int* code) {
  *code = HX_ERR_INVALID_ARG;
  if (!c) return "null config";
  if (c->ndim < 1 || c->ndim > 3) return "ndim must be 1, 2 or 3";
  if (c->coords != HX_CARTESIAN && c->coords != HX_SPHERICAL) return "unknown coordinate system";
  if (c->eos != HX_EOS_IDEAL && c->eos != HX_EOS_GAS_RADIATION) { *code = HX_ERR_UNSUPPORTED; return "unknown equation of state"; }
  if (c->eos == HX_EOS_GAS_RADIATION && (!(c->eos_R > 0.0) || !(c->eos_ar > 0.0))) return "gas + radiation EOS needs eos_R > 0 and eos_ar > 0";
  if (!(c->gamma > 1.0)) return "gamma must be > 1";
  if (c->riemann != HX_RIEMANN_HLL && c->riemann != HX_RIEMANN_HLLC) return "unknown Riemann solver";
  if (c->limiter < HX_LIM_NONE || c->limiter > HX_LIM_MC) return "unknown limiter";
  if (c->n_scalars < 0 || 2 + c->ndim + c->n_scalars > NVMAX) return "too many passive scalars";
  if (c->gravity < HX_GRAV_NONE || c->gravity > HX_GRAV_SELF) return "unknown gravity type";
  if (!(c->emon_eps >= 0.0)) return "emon_eps must be >= 0";
  if ((c->gravity == HX_GRAV_POINT_MASS || c->gravity == HX_GRAV_SELF) && c->coords != HX_SPHERICAL)
    return "point-mass gravity and self-gravity need spherical coordinates";
  for (int d = 0; d < 3; ++d) {
    if (d >= c->ndim) {
      if (c->n[d] != 1) return "inactive directions must have n = 1";
      continue;
    }
    if (c->n[d] < NG) return "active directions need at least 2 cells";
    if (c->bc_lo[d] < 0 || c->bc_lo[d] > HX_BC_WEDGE || c->bc_hi[d] < 0 || c->bc_hi[d] > HX_BC_WEDGE) return "unknown boundary condition";
    if ((c->bc_lo[d] == HX_BC_PERIODIC) != (c->bc_hi[d] == HX_BC_PERIODIC)) return "periodic must be set on both sides";
    if (c->coords == HX_SPHERICAL && d == 0 && c->bc_lo[d] == HX_BC_PERIODIC) return "the radial direction cannot be periodic";
    if (c->spacing[d] == HX_SPACING_CUSTOM) {
      if (!c->faces[d]) return "custom spacing needs a face array";
      for (int i = 0; i < c->n[d]; ++i)
        if (!(c->faces[d][i + 1] > c->faces[d][i])) return "face coordinates must increase strictly";
    } else if (c->spacing[d] == HX_SPACING_UNIFORM || c->spacing[d] == HX_SPACING_LOG) {
      if (!(c->hi[d] > c->lo[d])) return "hi must exceed lo";
      if (c->spacing[d] == HX_SPACING_LOG && !(c->lo[d] > 0.0)) return "logarithmic spacing needs lo > 0";
    } else {
      return "unknown spacing";
    }
  }
  *code = HX_OK;
  return nullptr;
}

// Padded face coordinates of one axis: interior faces, then ghost faces by copying cell widths
// from the far side (periodic) or mirroring them about the boundary (otherwise).
std::vector<double> padded_faces(const hx_config& c, int d, int ng) {
  const double PI = 3.14159265358979323846;
  const int n = c.n[d];
  std::vector<double> xf(n + 2 * ng + 1, 0.0);
  double* f = xf.data() + ng;
  if (ng == 0) {   // inactive direction: one cell spanning the given (or default) extent
    double lo = c.lo[d], hi = c.hi[d];
    if (!(hi > lo)) {
      lo = 0.0;
      hi = (c.coords == HX_SPHERICAL) ? (d == 1 ? PI : 2.0 * PI) : 1.0;
    }
    f[0] = lo;
    f[1] = hi;
    return xf;
  }
  if (c.spacing[d] == HX_SPACING_CUSTOM) {
    for (int i = 0; i <= n; ++i) f[i] = c.faces[d][i];
  } else if (c.spacing[d] == HX_SPACING_LOG) {
    const double ratio = c.hi[d] / c.lo[d];
    for (int i = 0; i <= n; ++i) f[i] = c.lo[d] * std::pow(ratio, (double)i / (double)n);
    f[0] = c.lo[d];
    f[n] = c.hi[d];
  } else {
    const double h = (c.hi[d] - c.lo[d]) / (double)n;
    for (int i = 0; i <= n; ++i) f[i] = c.lo[d] + (double)i * h;
    f[n] = c.hi[d];
  }
  for (int g = 1; g <= ng; ++g) {
    const double wlo = (c.bc_lo[d] == HX_BC_PERIODIC) ? f[n - g + 1] - f[n - g] : f[g] - f[g - 1];
    f[-g] = f[-g + 1] - wlo;
    const double whi = (c.bc_hi[d] == HX_BC_PERIODIC) ? f[g] - f[g - 1] : f[n - g + 1] - f[n - g];
    f[n + g] = f[n + g - 1] + whi;
  }
  return xf;
}

// Build every 1-D table on the host, upload once, and point h->T into the device block.
int build_tables(hx_handle* h) {
  const hx_config& c = h->cfg;
  const Layout& L = h->L;
  const bool sph = c.coords == HX_SPHERICAL;
  std::vector<double> xf[3];
  for (int d = 0; d < 3; ++d) xf[d] = padded_faces(c, d, L.ng[d]);

  std::vector<double> pool;
  auto reserve = [&](int d) {   // one table along axis d, returns its offset in the pool
    const size_t o = pool.size();
    pool.resize(o + (size_t)L.np[d], 1.0);
    return o;
  };
  size_t ones[3], iw[3], idx[3], hw[3], grav[3];
  for (int d = 0; d < 3; ++d) {
    ones[d] = reserve(d);
    iw[d] = reserve(d);
    idx[d] = reserve(d);
    hw[d] = reserve(d);
    grav[d] = reserve(d);
    for (int p = 0; p < L.np[d]; ++p) {
      const double lo = xf[d][p], hi = xf[d][p + 1];
      pool[iw[d] + p] = 1.0 / (hi - lo);
      pool[hw[d] + p] = 0.5 * (hi - lo);
      if (p >= 1) pool[idx[d] + p] = 1.0 / (0.5 * (lo + hi) - 0.5 * (xf[d][p - 1] + xf[d][p]));
      pool[grav[d] + p] = 0.0;
    }
  }
  // gravity seen by each cell of each active axis, mirrored behind reflecting faces (R25)
  auto g_raw = [&](int d, int idx_int) -> double {
    if (c.gravity == HX_GRAV_UNIFORM) return c.g[d];
    if ((c.gravity == HX_GRAV_POINT_MASS || c.gravity == HX_GRAV_SELF) && d == 0) {   // self-gravity: start value, rewritten every step
      const int p = idx_int + L.ng[0];
      const double rc = 0.5 * (xf[0][p] + xf[0][p + 1]);
      return -c.GM / (rc * rc);
    }
    return 0.0;
  };
  for (int d = 0; d < c.ndim; ++d) {
    const int n = c.n[d];
    for (int p = 0; p < L.np[d]; ++p) {
      const int i = p - L.ng[d];
      double g;
      if (i < 0) g = reflecting(c.bc_lo[d]) ? -g_raw(d, -1 - i) : (c.bc_lo[d] == HX_BC_PERIODIC ? g_raw(d, i + n) : g_raw(d, i));
      else if (i >= n) g = reflecting(c.bc_hi[d]) ? -g_raw(d, 2 * n - 1 - i) : (c.bc_hi[d] == HX_BC_PERIODIC ? g_raw(d, i - n) : g_raw(d, i));
      else g = g_raw(d, i);
      pool[grav[d] + p] = (c.gravity == HX_GRAV_NONE) ? 0.0 : g;
    }
  }
  size_t ar_m = 0, ar_p = 0, cr = 0, gr = 0, Ar = 0, rr = 0, irc = 0, idr = 0;
  size_t bt_m = 0, bt_p = 0, gt = 0, At = 0, st = 0, dthc = 0, idth = 0, isinc = 0, idphi = 0;
  if (sph) {
    ar_m = reserve(0); ar_p = reserve(0); cr = reserve(0); gr = reserve(0); Ar = reserve(0); rr = reserve(0); irc = reserve(0); idr = reserve(0);
    for (int p = 0; p < L.np[0]; ++p) {
      const double rm = xf[0][p], rp = xf[0][p + 1];
      const double v3 = (rp * rp * rp - rm * rm * rm) / 3.0, v2 = (rp * rp - rm * rm) / 2.0;
      pool[ar_m + p] = rm * rm / v3;
      pool[ar_p + p] = rp * rp / v3;
      pool[cr + p] = v2 / v3;
      pool[gr + p] = (rp * rp - rm * rm) / (2.0 * v3);
      pool[rr + p] = (rp - rm) / (rp + rm);
      pool[Ar + p] = (rp - rm) / (rp + rm) * ((rp * rp + rm * rm) / v3);
      pool[irc + p] = 1.0 / (0.5 * (rp + rm));
      pool[idr + p] = 1.0 / (rp - rm);
    }
    bt_m = reserve(1); bt_p = reserve(1); gt = reserve(1); At = reserve(1); st = reserve(1); dthc = reserve(1); idth = reserve(1); isinc = reserve(1);
    for (int p = 0; p < L.np[1]; ++p) {
      const double tm = xf[1][p], tp = xf[1][p + 1];
      const double dcos = std::cos(tm) - std::cos(tp), sm = std::sin(tm), sp = std::sin(tp);
      pool[bt_m + p] = sm / dcos;
      pool[bt_p + p] = sp / dcos;
      pool[gt + p] = (sp - sm) / dcos;
      pool[st + p] = (sp - sm) / (sp + sm);
      pool[At + p] = (sp - sm) / (sp + sm) * ((sp + sm) / dcos);
      pool[dthc + p] = (tp - tm) / dcos;
      pool[idth + p] = 1.0 / (tp - tm);
      pool[isinc + p] = 1.0 / std::sin(0.5 * (tm + tp));
    }
    idphi = reserve(2);
    for (int p = 0; p < L.np[2]; ++p) pool[idphi + p] = 1.0 / (xf[2][p + 1] - xf[2][p]);
  }

  size_t xfo[3];
  for (int d = 0; d < 3; ++d) {   // padded face coordinates (self-gravity kernels)
    xfo[d] = pool.size();
    pool.insert(pool.end(), xf[d].begin(), xf[d].end());
  }
  // Bitwise-uniform Cartesian grid (e.g. 2^k cells on a dyadic extent): every cell of an axis has the same
  // hw, 1/width and 1/(centre distance), so the step kernel may take them as constants without changing a bit.
  h->uniform = !sph && c.ndim >= 2;
  for (int d = 0; d < c.ndim && h->uniform; ++d) {
    for (int p = 1; p < L.np[d]; ++p)
      if (memcmp(&pool[hw[d] + p], &pool[hw[d]], 8) || memcmp(&pool[iw[d] + p], &pool[iw[d]], 8) ||
          memcmp(&pool[idx[d] + p], &pool[idx[d] + 1], 8))
        h->uniform = false;
    h->uni[d] = pool[hw[d] + 1] * pool[idx[d] + 1];
    h->uni[3 + d] = pool[iw[d] + 1];
  }

  const size_t bytes = pool.size() * sizeof(double);
  cudaError_t e = cudaMalloc(&h->d_tables, bytes);
  if (e != cudaSuccess) return cuda_fail(h, e, "cudaMalloc(tables)");
  e = cudaMemcpy(h->d_tables, pool.data(), bytes, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) return cuda_fail(h, e, "cudaMemcpy(tables)");
  const double* base = h->d_tables;
  for (int d = 0; d < 3; ++d) h->d_xf[d] = base + xfo[d];
  h->d_grav_r = h->d_tables + grav[0];
  Tables& T = h->T;
  for (int d = 0; d < 3; ++d) {
    for (int s = 0; s < 2; ++s)
      for (int e2 = 0; e2 < 3; ++e2) T.cf[d][s][e2] = base + ((!sph && e2 == d) ? iw[d] : ones[e2]);
    for (int e2 = 0; e2 < 3; ++e2) T.lf[d][e2] = base + ((!sph && e2 == d) ? iw[d] : ones[e2]);
    T.idx[d] = base + idx[d];
    T.hw[d] = base + hw[d];
    T.grav[d] = base + grav[d];
  }
  T.gr = T.Ar = T.rr = T.cr = base + ones[0];
  T.gt = T.At = T.st = base + ones[1];
  if (sph) {
    T.cf[0][0][0] = base + ar_m;
    T.cf[0][1][0] = base + ar_p;
    for (int s = 0; s < 2; ++s) {
      T.cf[1][s][0] = base + cr;
      T.cf[2][s][0] = base + cr;
      T.cf[2][s][1] = base + dthc;
      T.cf[2][s][2] = base + idphi;
    }
    T.cf[1][0][1] = base + bt_m;
    T.cf[1][1][1] = base + bt_p;
    T.lf[0][0] = base + idr;
    T.lf[1][0] = base + irc;
    T.lf[1][1] = base + idth;
    T.lf[2][0] = base + irc;
    T.lf[2][1] = base + isinc;
    T.lf[2][2] = base + idphi;
    T.gr = base + gr; T.Ar = base + Ar; T.rr = base + rr; T.cr = base + cr;
    T.gt = base + gt; T.At = base + At; T.st = base + st;
  }
  return HX_OK;
}

// Collect the event pair of the last timed step-kernel launch (call only after a stream sync).
void collect_timing(hx_handle* h) {
  if (!h->ev_pending) return;
  float ms = 0.f;
  if (cudaEventElapsedTime(&ms, h->ev0, h->ev1) == cudaSuccess) {
    h->kernel_ms += ms;
    h->kernel_launches++;
  }
  h->ev_pending = false;
}

StepArgs make_args(hx_handle* h, double dt) {
  StepArgs a;
  a.L = h->L;
  a.T = h->T;
  a.P = h->P;
  a.Uin = h->d_U[h->cur];
  a.Uout = h->d_U[1 - h->cur];
  a.dt = dt;
  a.rate_bits = &h->d_scal->rate_bits;
  a.status = &h->d_scal->status;
  return a;
}

}  // namespace

extern "C" {

const char* hx_version(void) { return "hx 0.2 (sm_100a)"; }
int hx_config_size(void) { return (int)sizeof(hx_config); }

int hx_create(const hx_config* cfg, hx_handle** out) {
  if (!out) return HX_ERR_INVALID_ARG;
  *out = nullptr;
  int code;
  const char* why = check_config(cfg, &code);
  if (why) return code;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return HX_ERR_CUDA;   // no CPU fallback
  hx_handle* h = new (std::nothrow) hx_handle();
  if (!h) return HX_ERR_ALLOC;
  h->cfg = *cfg;
  Layout& L = h->L;
  L.ndim = cfg->ndim;
  L.nvar = 2 + cfg->ndim + cfg->n_scalars;
  for (int d = 0; d < 3; ++d) {
    L.n[d] = cfg->n[d];
    L.ng[d] = d < cfg->ndim ? NG : 0;
    L.np[d] = L.n[d] + 2 * L.ng[d];
  }
  // Row pitch: multiple of 16 doubles (128 B) so every row starts on a cache line and TMA strides
  // are 16-byte multiples; `lead` shifts the first interior cell of each row onto a 128 B boundary.
  L.lead = (16 - (L.ng[0] % 16)) % 16;
  L.sy = ((long long)L.np[0] + L.lead + 15) / 16 * 16;
  L.sz = L.sy * L.np[1];
  L.sv = L.sz * L.np[2];
  h->P.gamma = cfg->gamma;
  h->P.gm1 = cfg->gamma - 1.0;
  h->P.igm1 = 1.0 / (cfg->gamma - 1.0);
  h->P.limiter = cfg->limiter;
  h->P.riemann = cfg->riemann;
  h->P.gravity = cfg->gravity;
  h->P.spherical = cfg->coords == HX_SPHERICAL;
  h->P.eos = cfg->eos;
  h->P.rgas = cfg->eos_R;
  h->P.arad = cfg->eos_ar;
  h->P.emon_eps = cfg->emon_eps > 0.0 ? cfg->emon_eps : 0.0;

  const size_t bytes = (size_t)L.nvar * (size_t)L.sv * sizeof(double);
  cudaError_t e;
  for (int b = 0; b < 2; ++b) {
    e = cudaMalloc(&h->d_U[b], bytes);
    if (e != cudaSuccess) { hx_destroy(h); return HX_ERR_ALLOC; }
    e = cudaMemset(h->d_U[b], 0, bytes);
    if (e != cudaSuccess) { hx_destroy(h); return HX_ERR_CUDA; }
  }
  e = cudaMalloc(&h->d_scal, sizeof(DevScalars));
  if (e == cudaSuccess) e = cudaMemset(h->d_scal, 0, sizeof(DevScalars));
  if (e == cudaSuccess) e = cudaMallocHost(&h->h_scal, sizeof(DevScalars));
  if (e != cudaSuccess) { hx_destroy(h); return HX_ERR_ALLOC; }
  if (cudaStreamCreateWithFlags(&h->side, cudaStreamNonBlocking) != cudaSuccess ||
      cudaEventCreateWithFlags(&h->ev_step, cudaEventDisableTiming) != cudaSuccess) { hx_destroy(h); return HX_ERR_CUDA; }
  const int rc = build_tables(h);
  if (rc != HX_OK) { hx_destroy(h); return rc; }
  if (cfg->gravity == HX_GRAV_SELF) {
    const long long rows = (long long)L.n[1] * L.n[2];
    h->sg_groups = (int)(rows < 296 ? rows : 296);
    if (cudaMalloc(&h->d_sg_partial, ((size_t)h->sg_groups * L.n[0] + L.n[1] + L.n[2]) * sizeof(double)) != cudaSuccess) { hx_destroy(h); return HX_ERR_ALLOC; }
  }
  h->cfg.faces[0] = h->cfg.faces[1] = h->cfg.faces[2] = nullptr;   // caller arrays are not retained
  *out = h;
  return HX_OK;
}

int hx_destroy(hx_handle* h) {
  if (!h) return HX_OK;
  if (h->plan2) tile2_plan_destroy(h->plan2);
  if (h->side) cudaStreamDestroy(h->side);
  if (h->ev_step) cudaEventDestroy(h->ev_step);
  if (h->ev0) cudaEventDestroy(h->ev0);
  if (h->ev1) cudaEventDestroy(h->ev1);
  for (int b = 0; b < 2; ++b)
    if (h->d_U[b]) cudaFree(h->d_U[b]);
  if (h->d_sg_partial) cudaFree(h->d_sg_partial);
  if (h->d_tables) cudaFree(h->d_tables);
  if (h->d_scal) cudaFree(h->d_scal);
  if (h->h_scal) cudaFreeHost(h->h_scal);
  delete h;
  return HX_OK;
}

int hx_set_stream(hx_handle* h, void* cuda_stream) {
  if (!h) return HX_ERR_INVALID_ARG;
  h->stream = (cudaStream_t)cuda_stream;
  return HX_OK;
}

int hx_set_option(hx_handle* h, int option, int value) {
  if (!h) return HX_ERR_INVALID_ARG;
  if (option == HX_OPT_KERNEL) {
    if (value < HX_KERNEL_AUTO || value > HX_KERNEL_TILED) return fail(h, HX_ERR_INVALID_ARG, "unknown kernel selection");
    if (value == HX_KERNEL_TILED && !tile2_supported(h->L, h->P)) return fail(h, HX_ERR_UNSUPPORTED, "the tiled kernel does not cover this configuration");
    h->kernel_opt = value;
    return HX_OK;
  }
  if (option == HX_OPT_ASYNC_HOST) {
    h->async_host = value != 0;
    return HX_OK;
  }
  if (option == HX_OPT_TIMING) {
    if (value && !h->ev0) {
      if (cudaEventCreate(&h->ev0) != cudaSuccess || cudaEventCreate(&h->ev1) != cudaSuccess) return fail(h, HX_ERR_CUDA, "cudaEventCreate");
    }
    h->timing = value != 0;
    return HX_OK;
  }
  return fail(h, HX_ERR_INVALID_ARG, "unknown option");
}

int hx_kernel_time(hx_handle* h, double* total_ms, long long* launches) {
  if (!h || !total_ms || !launches) return HX_ERR_INVALID_ARG;
  *total_ms = h->kernel_ms;
  *launches = h->kernel_launches;
  return HX_OK;
}

int hx_nvar(const hx_handle* h) { return h ? h->L.nvar : HX_ERR_INVALID_ARG; }
long long hx_launch_count(const hx_handle* h) { return h ? h->launches : 0; }
const char* hx_step_kernel_name(const hx_handle* h) { return h ? h->last_kernel : ""; }
const char* hx_last_error(const hx_handle* h) { return h ? h->err : "null handle"; }

int hx_set_state(hx_handle* h, const double* data, int mem_space, int form) {
  if (!h || !data) return HX_ERR_INVALID_ARG;
  if ((mem_space != HX_HOST && mem_space != HX_DEVICE) || (form != HX_CONSERVED && form != HX_PRIMITIVE))
    return fail(h, HX_ERR_INVALID_ARG, "bad mem_space or form");
  const Layout& L = h->L;
  const size_t nint = (size_t)L.n[0] * L.n[1] * L.n[2] * L.nvar;
  const double* src = data;
  cudaError_t e;
  if (mem_space == HX_HOST) {   // stage through the idle state buffer: no extra device memory
    double* stage = h->d_U[1 - h->cur];
    e = cudaMemcpyAsync(stage, data, nint * sizeof(double), cudaMemcpyHostToDevice, h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "hx_set_state: H2D copy");
    src = stage;
  }
  e = launch_pack(L, h->P, src, h->d_U[h->cur], form == HX_PRIMITIVE, h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "hx_set_state: pack kernel");
  h->launches++;
  e = cudaMemsetAsync(h->d_scal, 0, sizeof(DevScalars), h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "hx_set_state: memset");
  h->rate_valid = false;
  h->ghosts_valid = false;
  if (mem_space == HX_HOST && !h->async_host) {
    e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "hx_set_state: sync");
  }
  return HX_OK;
}

int hx_sync(hx_handle* h) {
  if (!h) return HX_ERR_INVALID_ARG;
  cudaError_t e = cudaMemcpyAsync(h->h_scal, h->d_scal, sizeof(DevScalars), cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "hx_sync");
  collect_timing(h);
  if (h->h_scal->status & 1) return fail(h, HX_ERR_NONPHYSICAL, "non-physical state (rho <= 0, P <= 0 or non-finite)");
  return HX_OK;
}

int hx_get_state(hx_handle* h, double* data, int mem_space, int form) {
  if (!h || !data) return HX_ERR_INVALID_ARG;
  if ((mem_space != HX_HOST && mem_space != HX_DEVICE) || (form != HX_CONSERVED && form != HX_PRIMITIVE))
    return fail(h, HX_ERR_INVALID_ARG, "bad mem_space or form");
  const Layout& L = h->L;
  const size_t nint = (size_t)L.n[0] * L.n[1] * L.n[2] * L.nvar;
  double* dst = (mem_space == HX_HOST) ? h->d_U[1 - h->cur] : data;
  cudaError_t e = launch_unpack(L, h->P, h->d_U[h->cur], dst, form == HX_PRIMITIVE, h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "hx_get_state: unpack kernel");
  h->launches++;
  if (mem_space == HX_HOST) {
    e = cudaMemcpyAsync(data, dst, nint * sizeof(double), cudaMemcpyDeviceToHost, h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "hx_get_state: D2H copy");
  }
  if (mem_space == HX_HOST && h->async_host) return HX_OK;   // enqueued only: the caller synchronises with hx_sync
  e = cudaMemcpyAsync(h->h_scal, h->d_scal, sizeof(DevScalars), cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "hx_get_state: sync");
  collect_timing(h);
  if (h->h_scal->status & 1) return fail(h, HX_ERR_NONPHYSICAL, "non-physical state (rho <= 0, P <= 0 or non-finite)");
  return HX_OK;
}

int hx_compute_dt(hx_handle* h, double cfl, double* dt_out) {
  if (!h || !dt_out) return HX_ERR_INVALID_ARG;
  if (!(cfl > 0.0)) return fail(h, HX_ERR_INVALID_ARG, "cfl must be positive");
  cudaError_t e;
  bool ran_rate_kernel = false;
  if (!h->rate_valid) {
    ran_rate_kernel = true;
    e = cudaMemsetAsync(&h->d_scal->rate_bits, 0, sizeof(unsigned long long), h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "hx_compute_dt: memset");
    e = launch_rate(h->L, h->T, h->P, h->d_U[h->cur], &h->d_scal->rate_bits, &h->d_scal->status, h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "hx_compute_dt: rate kernel");
    h->launches++;
    h->rate_valid = true;
  }
  if (ran_rate_kernel) {
    e = cudaMemcpyAsync(h->h_scal, h->d_scal, sizeof(DevScalars), cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  } else {
    // the rate was folded in by the last step kernel: read it back on the side stream, which waits for that kernel
    // only, so the ghost fill hx_step already queued for the next step keeps the GPU busy meanwhile
    e = cudaStreamWaitEvent(h->side, h->ev_step, 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h->h_scal, h->d_scal, sizeof(DevScalars), cudaMemcpyDeviceToHost, h->side);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->side);
  }
  if (e != cudaSuccess) return cuda_fail(h, e, "hx_compute_dt: sync");
  collect_timing(h);
  if (h->h_scal->status & 1) return fail(h, HX_ERR_NONPHYSICAL, "non-physical state (rho <= 0, P <= 0 or non-finite)");
  double rate;
  memcpy(&rate, &h->h_scal->rate_bits, sizeof(double));
  if (!(rate > 0.0) || !std::isfinite(rate)) return fail(h, HX_ERR_NONPHYSICAL, "CFL rate is not positive and finite");
  *dt_out = cfl / rate;
  return HX_OK;
}

// Diagnostic: the handle path of the self-gravity refresh (the same launch hx_step makes), table read back.
int hx_self_gravity_table(hx_handle* h, double* out, int mem_space) {
  if (!h || !out) return HX_ERR_INVALID_ARG;
  if (mem_space != HX_HOST && mem_space != HX_DEVICE) return fail(h, HX_ERR_INVALID_ARG, "bad mem_space");
  if (h->cfg.gravity != HX_GRAV_SELF) return fail(h, HX_ERR_UNSUPPORTED, "hx_self_gravity_table needs HX_GRAV_SELF");
  const Layout& L = h->L;
  cudaError_t e = launch_self_gravity(L, h->d_U[h->cur], h->d_xf, h->d_sg_partial, h->sg_groups, h->d_grav_r, h->cfg.GM, h->cfg.G,
                                      h->cfg.bc_lo[0], h->cfg.bc_hi[0], h->d_sg_partial + (size_t)h->sg_groups * L.n[0], &h->sg_weights_ready,
                                      h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "hx_self_gravity_table: self-gravity");
  h->launches += 2;
  e = cudaMemcpyAsync(out, h->d_grav_r + L.ng[0], (size_t)L.n[0] * sizeof(double),
                      mem_space == HX_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, h->stream);
  if (e == cudaSuccess && mem_space == HX_HOST) e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "hx_self_gravity_table: copy");
  return HX_OK;
}

int hx_step(hx_handle* h, double dt) {
  if (!h) return HX_ERR_INVALID_ARG;
  if (!(dt > 0.0) || !std::isfinite(dt)) return fail(h, HX_ERR_INVALID_ARG, "dt must be positive and finite");
  const Layout& L = h->L;
  cudaError_t e;
  if (!h->ghosts_valid) {   // A0: all directions, one launch (normally done eagerly at the end of the previous hx_step)
    e = launch_ghost_fill(L, h->d_U[h->cur], h->cfg.bc_lo, h->cfg.bc_hi, 0, h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "hx_step: ghost fill");
    h->launches++;
  }
  if (h->cfg.gravity == HX_GRAV_SELF) {   // Eq. 4 from U^n: shell masses, scan over r, new radial acceleration table
    e = launch_self_gravity(L, h->d_U[h->cur], h->d_xf, h->d_sg_partial, h->sg_groups, h->d_grav_r, h->cfg.GM, h->cfg.G, h->cfg.bc_lo[0],
                            h->cfg.bc_hi[0], h->d_sg_partial + (size_t)h->sg_groups * L.n[0], &h->sg_weights_ready, h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "hx_step: self-gravity");
    h->launches += 2;
  }
  e = cudaMemsetAsync(&h->d_scal->rate_bits, 0, sizeof(unsigned long long), h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "hx_step: memset");
  StepArgs a = make_args(h, dt);
  bool use_tile2 = false;
  const int ko = h->kernel_opt;
  if ((ko == HX_KERNEL_AUTO || ko == HX_KERNEL_TILED) && tile2_supported(L, h->P)) {
    if (!h->plan2 && !h->plan2_tried) {
      h->plan2_tried = true;
      const int grav_z = h->cfg.gravity == HX_GRAV_UNIFORM && h->cfg.g[0] == 0.0 && h->cfg.g[1] == 0.0;
      e = tile2_plan_create(L, h->P, h->d_U, h->uniform ? h->uni : nullptr, grav_z, h->cfg.bc_lo[0], h->cfg.bc_hi[0], &h->plan2);
      if (e != cudaSuccess) {
        h->plan2 = nullptr;
        return cuda_fail(h, e, "hx_step: tile2 plan");   // no silent fallback to a slower path
      }
    }
    use_tile2 = h->plan2 != nullptr;
    if (!use_tile2) return fail(h, HX_ERR_CUDA, "tile2 kernel unavailable");
  }
  const bool timed = h->timing && !h->ev_pending;
  if (timed) cudaEventRecord(h->ev0, h->stream);
  if (use_tile2) {
    e = launch_step_tile2(h->plan2, a, h->cur, h->stream);
    h->last_kernel = tile2_kernel_name(h->plan2);
  } else {
    e = launch_step_generic(a, h->stream);
    h->last_kernel = "generic";
  }
  if (e != cudaSuccess) return cuda_fail(h, e, "hx_step: step kernel");
  if (timed) {
    cudaEventRecord(h->ev1, h->stream);
    h->ev_pending = true;
  }
  h->launches++;
  h->cur = 1 - h->cur;
  h->rate_valid = true;
  // The next step needs the ghost layers of the new state whatever its dt will be: fill them now, behind the event
  // hx_compute_dt waits for, so that the host's read-back of the CFL rate overlaps this kernel.
  e = cudaEventRecord(h->ev_step, h->stream);
  if (e == cudaSuccess)   // (the 3-D tile kernel has written the x-ghost cells of the interior rows itself)
    e = launch_ghost_fill(L, h->d_U[h->cur], h->cfg.bc_lo, h->cfg.bc_hi, use_tile2 && tile2_writes_x_ghosts(h->plan2), h->stream);
  if (e != cudaSuccess) return cuda_fail(h, e, "hx_step: eager ghost fill");
  h->launches++;
  h->ghosts_valid = true;
  return HX_OK;
}

}  // extern "C"

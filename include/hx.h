/*
 * hx.h -- C ABI of the B200-native fp64 Godunov finite-volume hydro step
 * (hot path of HERACLES++, arxiv 2503.04428; Sect. 2-3).
 *
 * One handle = one logically Cartesian block on one GPU (Sect. 3.1.1).  The library
 * owns every device allocation: the double-buffered conserved state, stored as structure-of-arrays
 * fp64 [nvar][n2+4][n1+4][pitch0] with two ghost layers per face in active directions, and the 1-D
 * geometry tables.  Caller buffers are only read or written during hx_set_state / hx_get_state;
 * nothing is retained.  All calls are host functions; kernels run on the handle's stream.
 *
 * Caller state buffers are interior-only structure-of-arrays [nvar][n2][n1][n0], direction 0
 * fastest, nvar = 2 + ndim + n_scalars, field order
 *     HX_CONSERVED: rho, m_0..m_{ndim-1}, E, rho*f_1..rho*f_ns          (Eq. 1a-1d)
 *     HX_PRIMITIVE: rho, u_0..u_{ndim-1}, P, f_1..f_ns                  (Eq. 5)
 * Directions are (x,y,z) or, with HX_SPHERICAL, (r,theta,phi) (L145).
 *
 * Errors: every function returns HX_OK or a negative code; nothing throws, exits or prints.
 * hx_last_error() gives a message for the last failing call on that handle.  There is no CPU
 * fallback: without a CUDA device hx_create fails with HX_ERR_CUDA.
 */
#ifndef HX_H
#define HX_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct hx_handle hx_handle;

enum { HX_OK = 0, HX_ERR_INVALID_ARG = -1, HX_ERR_ALLOC = -2, HX_ERR_CUDA = -3,
       HX_ERR_NONPHYSICAL = -4 /* rho<=0, P<=0 or non-finite seen */, HX_ERR_UNSUPPORTED = -5 };
enum { HX_CARTESIAN = 0, HX_SPHERICAL = 1 };
/* Boundary conditions (periodic, null gradient, reflective).  HX_BC_WEDGE is the
 * reflective condition on the angular faces of a spherical wedge (L424). */
enum { HX_BC_PERIODIC = 0, HX_BC_TRANSMISSIVE = 1, HX_BC_REFLECTING = 2, HX_BC_WEDGE = 3 };
enum { HX_EOS_IDEAL = 0 /* Eq. 5 */, HX_EOS_GAS_RADIATION = 1 /* Eq. 6-7: ideal gas in equilibrium with radiation */ };
enum { HX_RIEMANN_HLL = 0, HX_RIEMANN_HLLC = 1 };       /* L201 */
/* Slope limiters (L189) + first order (HX_LIM_NONE) + monotonised central (BASELINE.json configs) */
enum { HX_LIM_NONE = 0, HX_LIM_MINMOD = 1, HX_LIM_VANLEER = 2, HX_LIM_VANALBADA = 3, HX_LIM_MC = 4 };
enum { HX_GRAV_NONE = 0, HX_GRAV_UNIFORM = 1 /* Eq. 2 */, HX_GRAV_POINT_MASS = 2 /* Eq. 3 */,
       HX_GRAV_SELF = 3 /* Eq. 4: central mass + spherically averaged mass of the grid inside r, refreshed every step */ };
enum { HX_SPACING_UNIFORM = 0, HX_SPACING_LOG = 1, HX_SPACING_CUSTOM = 2 };   /* L149 */
enum { HX_HOST = 0, HX_DEVICE = 1 };
enum { HX_CONSERVED = 0, HX_PRIMITIVE = 1 };
/* Step kernel selection (hx_set_option(HX_OPT_KERNEL, ..)): AUTO picks the fused tile kernel where
 * it applies and the generic one elsewhere; the other two force one path (tests, profiling). */
enum { HX_OPT_KERNEL = 0, HX_OPT_TIMING = 1 /* 0/1: bracket each step-kernel launch with CUDA events */,
       HX_OPT_ASYNC_HOST = 2 /* 0/1: hx_set_state / hx_get_state with HOST buffers only enqueue their copies (see below) */ };
enum { HX_KERNEL_AUTO = 0, HX_KERNEL_GENERIC = 1,
       HX_KERNEL_TILED = 2 /* the fused TMA-staged tile kernels ("tile2*" in 3-D, "tile2d*" on 2-D Cartesian grids): what AUTO picks where they apply */ };

#define HX_MAX_NVAR 16

typedef struct {
  int ndim;               /* 1, 2 or 3; active directions are 0..ndim-1                              */
  int coords;             /* HX_CARTESIAN or HX_SPHERICAL                                            */
  int n[3];               /* interior cells; inactive directions must be 1; active ones >= 2         */
  double lo[3], hi[3];    /* extents.  Inactive directions: Cartesian width hi-lo (1 if hi<=lo);     */
                          /* spherical theta defaults to [0,pi] and phi to [0,2pi] if hi<=lo         */
  int spacing[3];         /* per direction: uniform, logarithmic (lo>0) or custom                    */
  const double* faces[3]; /* HX_SPACING_CUSTOM: n[d]+1 strictly increasing HOST face coordinates,    */
                          /* copied during hx_create                                                 */
  int bc_lo[3], bc_hi[3]; /* periodic must be set on both sides of a direction                       */
  int eos;                /* HX_EOS_IDEAL or HX_EOS_GAS_RADIATION (T from e by Newton-Raphson, L102)         */
  double gamma;           /* adiabatic index > 1                                                     */
  int riemann, limiter, n_scalars;
  int gravity;            /* HX_GRAV_*; point mass and self-gravity need HX_SPHERICAL                */
  double g[3];            /* uniform: acceleration vector (force = +rho*g, R12)            */
  double GM;              /* point mass: g = -GM/r_c^2 e_r                                           */
  double eos_R;           /* HX_EOS_GAS_RADIATION: k_b / mu, gas constant per unit mass (Eq. 6a); > 0         */
  double eos_ar;          /* HX_EOS_GAS_RADIATION: radiation constant a_r (Eq. 6a-6b); > 0                    */
  double G;               /* HX_GRAV_SELF: gravitational constant (GM is then G times the central mass)      */
  double emon_eps;        /* > 0: monitoring of the internal energy (Eq. 10-12) with this epsilon (paper: 1e-6) */
} hx_config;

/* Validate cfg, allocate the padded double-buffered state and the geometry tables on the current
 * CUDA device.  *out is NULL on failure. */
int hx_create(const hx_config* cfg, hx_handle** out);
/* Free everything the handle owns.  NULL is accepted. */
int hx_destroy(hx_handle* h);
/* Use the given cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream) for all later work.
 * NULL = the legacy default stream.  The caller keeps ownership of the stream. */
int hx_set_stream(hx_handle* h, void* cuda_stream);
int hx_set_option(hx_handle* h, int option, int value);
/* Copy the caller's interior state in (mem_space = HX_HOST or HX_DEVICE pointer; form = conserved
 * or primitive, converted through the EOS).  Returns after the copy is enqueued (device pointer)
 * or finished (host pointer). */
int hx_set_state(hx_handle* h, const double* data, int mem_space, int form);
/* With HX_OPT_ASYNC_HOST = 1 the two calls above / below return as soon as their copies are enqueued on the handle's
 * stream when given a HOST pointer: the buffer must be page-locked and stay untouched until hx_sync (or any other
 * synchronising call) returns; hx_get_state then reports HX_ERR_NONPHYSICAL at that later call.  This lets the
 * host-to-device copy of one handle overlap the device-to-host copy of another on the full-duplex link. */
int hx_sync(hx_handle* h);
/* Copy the interior state out; synchronises the stream.  Returns HX_ERR_NONPHYSICAL (after
 * copying) if a kernel flagged a non-physical state since the last hx_set_state. */
int hx_get_state(hx_handle* h, double* data, int mem_space, int form);
/* A7: dt = cfl / max over interior cells of sum_d (|u_d|+c_s)/l_d (R2).  Uses the rate
 * the last hx_step folded into its update when available, else runs the reduction kernel.
 * One 16-byte device-to-host copy; waits for the last step kernel (not for the ghost fill hx_step queues behind it)
 * or, right after hx_set_state, for the reduction kernel. */
int hx_compute_dt(hx_handle* h, double cfl, double* dt_out);
/* A0-A6 (+A7 fused): ghost fill (done eagerly at the end of the previous hx_step when there was one), then one
 * unsplit MUSCL-Hancock / Godunov update of every interior cell by dt (Eq. 17-19, sources Eq. 13-16, gravity Eq. 2-3).  Asynchronous on the stream; device
 * side errors surface at the next hx_compute_dt / hx_get_state. */
int hx_step(hx_handle* h, double dt);
/* Number of stored fields, 2 + ndim + n_scalars. */
int hx_nvar(const hx_handle* h);
/* Name of the step kernel the last hx_step used ("generic", "tile2", "tile2_uni", "tile2_uni12", "tile2_rad", "tile2_rad_emon", "tile2_emon", "tile2_emon_uni", "tile2d", "tile2d_uni"). */
const char* hx_step_kernel_name(const hx_handle* h);
const char* hx_last_error(const hx_handle* h);
const char* hx_version(void);
/* ABI handshake for bindings: sizeof(hx_config) as this library was compiled.  A binding whose struct has another size
 * was written for another revision of this header and must not call hx_create. */
int hx_config_size(void);

/* ---- diagnostics and measurement hooks (bench.py, profiling); not needed to run the method ---------------------- */
/* Kernels launched by this handle so far (for bench.py's gpu_launches). */
long long hx_launch_count(const hx_handle* h);
/* With HX_OPT_TIMING on: device time (ms) spent in the step kernel alone, summed over the launches
 * measured so far, and their number.  Read after a synchronising call (hx_compute_dt / hx_get_state);
 * a launch whose events were not yet collected when the next step started is not counted. */
int hx_kernel_time(hx_handle* h, double* total_ms, long long* launches);
/* Device probe (no handle, default stream, synchronous): measured FP64 FMA throughput of the current
 * GPU in TFLOP/s (1 FMA = 2 flop; many independent chains on every SM) and the issue-to-issue latency
 * of a dependent DFMA in SM cycles.  This is the denominator of the "alu" roofline. */
int hx_probe_fp64(double* tflops, double* dep_latency_cycles);
/* HX_GRAV_SELF handles only: refresh the radial acceleration table from the CURRENT state exactly as hx_step does before its
 * step kernel (Eq. 4, R28; shell-mass reduction through the handle's cudaMalloc'ed scratch + scan) and copy its n[0]
 * interior entries g_r(r_c,i) to out (HX_HOST or HX_DEVICE pointer).  Synchronises for a host pointer.  HX_ERR_UNSUPPORTED for
 * other gravity types.  The cross-check of hx_self_gravity_noalloc below. */
int hx_self_gravity_table(hx_handle* h, double* out, int mem_space);

/* ---- entry point that allocates nothing (callers under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc) -- */
/* The self-gravity refresh of Eq. 4 (R28) without a handle and without any device allocation:
 *   g[i] = -( GM + G (4 pi / dOmega) ( sum_{i'<i} m_i' + m_i (r_c^3 - r_-^3)/(r_+^3 - r_-^3) ) ) / r_c^2,   i = 0 .. n0-1,
 * m_i = sum_{j,k} rho dV the shell masses, dOmega the solid angle of the grid, r_c = (r_- + r_+)/2.
 * ALL pointers are DEVICE pointers owned by the caller: rho = interior density [n2][n1][n0] (direction 0 fastest), faces_r /
 * faces_theta / faces_phi = n0+1 / n1+1 / n2+1 increasing face coordinates, g = n0 outputs.  The partial shell sums (the scratch
 * the handle path keeps in cudaMalloc'ed memory) live in a file-scope `static __device__` array of the library, 2 MiB + 32 KiB,
 * which every GPU that loads libhx.so holds until the process exits.  Hence the limits: n0 <= HX_NOALLOC_MAX_N0 and
 * n1 + n2 <= HX_NOALLOC_MAX_ANGULAR; larger sizes are rejected with HX_ERR_UNSUPPORTED (message from hx_noalloc_error()).
 * The call enqueues three kernels on cuda_stream (a cudaStream_t, NULL = legacy default stream) and returns; it calls no
 * cudaMalloc / cudaFree / allocating library routine and does not synchronise.  Every call on a GPU shares the one array: the
 * array keeps the last call's contents (each call overwrites every entry it later reads, nothing needs to start at zero), and
 * two calls that overlap on the GPU (different streams, different host threads) RACE on it -- serialise them. */
#define HX_NOALLOC_MAX_N0 2048
#define HX_NOALLOC_MAX_ANGULAR 4096
int hx_self_gravity_noalloc(const double* rho, const double* faces_r, const double* faces_theta, const double* faces_phi, int n0, int n1,
                            int n2, double GM, double G, double* g, void* cuda_stream);
/* Message of the last failing hx_self_gravity_noalloc call of this host thread ("" if none). */
const char* hx_noalloc_error(void);

#ifdef __cplusplus
}
#endif
#endif

/*
 * ox.h -- C interface of the CPU ORACLE for the Godunov finite-volume hydro step of
 * HERACLES++ (arxiv 2503.04428; Sect. 2-3, Eq. 1-5, 13-19).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA path (paper_2503_04428_b200/csrc, include/hx.h);
 * the struct below is declared here on its own on purpose.
 *
 * Everything is fp64, host memory only.  State buffers are interior-only
 * structure-of-arrays [nvar][n2][n1][n0] (direction 0 fastest), with
 * nvar = 2 + ndim + n_scalars and field order
 *   CONSERVED: rho, m_0..m_{ndim-1}, E, rho*f_1..rho*f_ns
 *   PRIMITIVE: rho, u_0..u_{ndim-1}, P, f_1..f_ns
 */
#ifndef OX_H
#define OX_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct ox_handle ox_handle;

enum { OX_OK = 0, OX_ERR_INVALID_ARG = -1, OX_ERR_ALLOC = -2, OX_ERR_NONPHYSICAL = -4, OX_ERR_UNSUPPORTED = -5 };
enum { OX_CARTESIAN = 0, OX_SPHERICAL = 1 };
enum { OX_BC_PERIODIC = 0, OX_BC_TRANSMISSIVE = 1, OX_BC_REFLECTING = 2, OX_BC_WEDGE = 3 };
enum { OX_EOS_IDEAL = 0 /* Eq. 5 */, OX_EOS_GAS_RADIATION = 1 /* Eq. 6-7: ideal gas in equilibrium with radiation */ };
enum { OX_RIEMANN_HLL = 0, OX_RIEMANN_HLLC = 1 };
enum { OX_LIM_NONE = 0, OX_LIM_MINMOD = 1, OX_LIM_VANLEER = 2, OX_LIM_VANALBADA = 3, OX_LIM_MC = 4 };
enum { OX_GRAV_NONE = 0, OX_GRAV_UNIFORM = 1, OX_GRAV_POINT_MASS = 2,
       OX_GRAV_SELF = 3 /* Eq. 4: central mass + spherically averaged mass of the grid inside r */ };
enum { OX_SPACING_UNIFORM = 0, OX_SPACING_LOG = 1, OX_SPACING_CUSTOM = 2 };
enum { OX_CONSERVED = 0, OX_PRIMITIVE = 1 };

typedef struct {
  int ndim;            /* 1, 2 or 3: active directions are 0..ndim-1                           */
  int coords;          /* OX_CARTESIAN: (x,y,z); OX_SPHERICAL: (r,theta,phi)                   */
  int n[3];            /* interior cells per direction; inactive directions must be 1          */
  double lo[3], hi[3]; /* extents; inactive: Cartesian width hi-lo (1 if hi<=lo); spherical    */
                       /* inactive theta defaults to [0,pi], phi to [0,2pi] if hi<=lo          */
  int spacing[3];
  const double* faces[3]; /* OX_SPACING_CUSTOM: n[d]+1 increasing face coordinates (copied)    */
  int bc_lo[3], bc_hi[3];
  int eos;
  double gamma;
  int riemann, limiter, n_scalars;
  int gravity;
  double g[3];         /* OX_GRAV_UNIFORM: acceleration vector                                  */
  double GM;           /* OX_GRAV_POINT_MASS: g = -GM/r_c^2 e_r (spherical only), Eq. 3         */
  double eos_R;        /* OX_EOS_GAS_RADIATION: k_b / mu (gas constant per unit mass), Eq. 6a     */
  double eos_ar;       /* OX_EOS_GAS_RADIATION: radiation constant a_r, Eq. 6a-6b                 */
  double G;            /* OX_GRAV_SELF: gravitational constant; GM is then G times the central mass M_c */
  double emon_eps;     /* > 0: internal-energy monitoring (Eq. 10-12) with this epsilon (paper: 1e-6); 0: off */
} ox_config;

int ox_create(const ox_config* cfg, ox_handle** out);
int ox_destroy(ox_handle* h);
int ox_nvar(const ox_handle* h);
int ox_set_state(ox_handle* h, const double* data, int form);
int ox_get_state(ox_handle* h, double* data, int form);
/* O7: dt = cfl / max_i sum_d (|u_d|+c_s)/l_d.  Returns OX_ERR_NONPHYSICAL if rho<=0, P<=0 or non-finite. */
int ox_compute_dt(ox_handle* h, double cfl, double* dt_out);
/* O0-O6, whole-array passes. */
int ox_step(ox_handle* h, double dt);
/* Deliberately naive second implementation: the update of ONE interior cell written straight from
 * O0-O6 with boundary conditions applied by index mapping (no ghost arrays, no stored intermediates).
 * Reads the current state, does not modify it.  out = nvar conserved values at t+dt. */
int ox_cell_update(ox_handle* h, int i, int j, int k, double dt, double* out);

/* Pieces exposed for the pins in tests/ ------------------------------------------------- */
/* Riemann flux in direction dir between two conserved states (length nvar = 2+ndim+ns). */
int ox_riemann_flux(int riemann, double gamma, int ndim, int ns, int dir, const double* UL, const double* UR, double* F);
/* Analytic flux F_dir(U). */
int ox_physical_flux(double gamma, int ndim, int ns, int dir, const double* U, double* F);
/* EOS closures for the pins: P(rho, e) (Eq. 5 / Eq. 6 through the Newton-Raphson solve for T, L102), e(rho, P),
 * c_s(rho, P) (Eq. 5 / Eq. 7).  eos = OX_EOS_*; R = k_b/mu and ar are ignored by the ideal gas. */
/* OX_GRAV_SELF: acceleration g_r(r_c) of interior radial cell i for the CURRENT state (for the pins). */
int ox_self_gravity(ox_handle* h, int i, double* g_out);
double ox_eos_pressure(int eos, double gamma, double R, double ar, double rho, double e);
double ox_eos_energy(int eos, double gamma, double R, double ar, double rho, double P);
double ox_eos_sound_speed(int eos, double gamma, double R, double ar, double rho, double P);
double ox_limiter(int limiter, double a, double b);
/* Geometry of interior or ghost cell (i,j,k): dV, dS[d][0 = minus face, 1 = plus face], centre xc[d]. */
int ox_cell_geometry(const ox_handle* h, int i, int j, int k, double* dV, double* dS6, double* xc3);
/* Padded face coordinates of direction d: n[d]+1+2*ng values (ng = 2 if active else 0). */
int ox_faces(const ox_handle* h, int d, double* out);
int ox_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif

"""Seeded synthetic workloads: the five BASELINE.json configurations (and reduced copies).

This module holds NO arithmetic of the method (no EOS, no fluxes, no limiter): it only writes
problem descriptions (plain dicts) and initial PRIMITIVE fields (rho, u_d, P, f_s) with numpy.
It is the one module shared by the CUDA path's tests/bench and by the CPU oracle's tests; it
imports neither of them.  The random numbers are a counter-based splitmix64 stream indexed by
the linear interior cell index, so the fields do not depend on generation order (DESIGN.md,
"Input recipe").

The configurations stand in for the paper's workloads (Sect. 4.1 KH, 4.2 RT, 4.3 /
App. C.4 Sedov, App. C.1 Sod, Sect. 5.5 supernova wedge); none of the paper's data files is used.
"""
import math

import numpy as np

# enum values shared by the problem descriptions (the CUDA header and the oracle header each declare the same numbers)
CARTESIAN, SPHERICAL = 0, 1
BC_PERIODIC, BC_TRANSMISSIVE, BC_REFLECTING, BC_WEDGE = 0, 1, 2, 3
RIEMANN_HLL, RIEMANN_HLLC = 0, 1
LIM_NONE, LIM_MINMOD, LIM_VANLEER, LIM_VANALBADA, LIM_MC = 0, 1, 2, 3, 4
GRAV_NONE, GRAV_UNIFORM, GRAV_POINT_MASS, GRAV_SELF = 0, 1, 2, 3
EOS_IDEAL, EOS_GAS_RADIATION = 0, 1
SPACING_UNIFORM, SPACING_LOG, SPACING_CUSTOM = 0, 1, 2

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def splitmix64(x: np.ndarray) -> np.ndarray:
    """One splitmix64 output per 64-bit counter value (vectorised, wraps modulo 2^64)."""
    with np.errstate(over="ignore"):
        z = (x.astype(np.uint64) + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return z ^ (z >> np.uint64(31))


def noise(seed: int, shape) -> np.ndarray:
    """Uniform noise in [-1, 1): u(idx) = 2*(splitmix64(seed ^ idx) >> 11)*2^-53 - 1, idx = linear index."""
    count = int(np.prod(shape))
    out = np.empty(count, dtype=np.float64)
    chunk = 1 << 24
    for start in range(0, count, chunk):
        idx = np.arange(start, min(count, start + chunk), dtype=np.uint64)
        bits = splitmix64(idx ^ np.uint64(seed)) >> np.uint64(11)
        out[start:start + idx.size] = 2.0 * (bits.astype(np.float64) * 2.0 ** -53) - 1.0
    return out.reshape(shape)


def uniform_faces(lo, hi, n):
    f = lo + np.arange(n + 1, dtype=np.float64) * ((hi - lo) / n)
    f[-1] = hi
    return f


def log_faces(lo, hi, n):
    f = lo * np.power(hi / lo, np.arange(n + 1, dtype=np.float64) / n)
    f[0], f[-1] = lo, hi
    return f


def centres(faces):
    return 0.5 * (faces[1:] + faces[:-1])


def _spec(name, ndim, n, faces, bc_lo, bc_hi, gamma, limiter, riemann=RIEMANN_HLLC, coords=CARTESIAN,
          n_scalars=0, gravity=GRAV_NONE, g=(0.0, 0.0, 0.0), GM=0.0, cfl=0.8, steps=1, t_end=None, seed=0,
          eos=EOS_IDEAL, eos_R=0.0, eos_ar=0.0, G=0.0, emon_eps=0.0):
    n3 = list(n) + [1] * (3 - len(n))
    return {
        "name": name, "ndim": ndim, "coords": coords, "n": n3,
        "lo": [float(f[0]) for f in faces] + [0.0] * (3 - len(faces)),
        "hi": [float(f[-1]) for f in faces] + [0.0] * (3 - len(faces)),
        "spacing": [SPACING_CUSTOM] * len(faces) + [SPACING_UNIFORM] * (3 - len(faces)),
        "faces": list(faces) + [None] * (3 - len(faces)),
        "bc_lo": list(bc_lo) + [0] * (3 - len(bc_lo)), "bc_hi": list(bc_hi) + [0] * (3 - len(bc_hi)),
        "eos": eos, "eos_R": eos_R, "eos_ar": eos_ar,
        "gamma": gamma, "riemann": riemann, "limiter": limiter, "n_scalars": n_scalars,
        "gravity": gravity, "g": list(g), "GM": GM, "G": G, "emon_eps": emon_eps,
        "cfl": cfl, "steps": steps, "t_end": t_end, "seed": seed,
        "nvar": 2 + ndim + n_scalars,
    }


def sod_1d(n=1000):
    """C1: PAPER.md App. C.1 (Eq. C.1) initial condition on n cells, transmissive, minmod + HLLC, CFL 0.8."""
    fx = uniform_faces(0.0, 1.0, n)
    spec = _spec("sod_1d", 1, [n], [fx], [BC_TRANSMISSIVE], [BC_TRANSMISSIVE], 1.4, LIM_MINMOD,
                 cfl=0.8, steps=None, t_end=0.2, seed=1001)
    x = centres(fx)
    W = np.empty((3, 1, 1, n))
    left = x < 0.5
    W[0, 0, 0] = np.where(left, 1.0, 0.125)
    W[1, 0, 0] = 0.0
    W[2, 0, 0] = np.where(left, 1.0, 0.1)
    return spec, W


def kh_2d(n=1024, seed=1002):
    """C2: 2-D periodic shear layer + 1 scalar, MC + HLLC, CFL 0.8, 200 steps (shape of PAPER.md Sect. 4.1)."""
    nx, ny = (n, n) if np.isscalar(n) else n
    fx = uniform_faces(0.0, 1.0, nx)
    fy = uniform_faces(0.0, 1.0, ny)
    spec = _spec("kh_2d", 2, [nx, ny], [fx, fy], [BC_PERIODIC] * 2, [BC_PERIODIC] * 2, 1.4, LIM_MC,
                 n_scalars=1, cfl=0.8, steps=200, seed=seed)
    y = centres(fy)
    band = (np.abs(y - 0.5) < 0.25)[:, None]
    W = np.empty((5, 1, ny, nx))
    W[0, 0] = np.where(band, 2.0, 1.0)
    W[1, 0] = np.where(band, 0.5, -0.5)
    W[2, 0] = 0.01 * noise(seed, (ny, nx))
    W[3, 0] = 2.5
    W[4, 0] = np.where(band, 1.0, 0.0)
    return spec, W


def sedov_3d(n=256, seed=1003):
    """C3: 3-D Cartesian blast, transmissive, gamma 5/3, minmod + HLLC, CFL 0.6, 100 steps
    (shape of PAPER.md Sect. 4.3 / App. C.4).  E = 1 as thermal energy in the cells whose
    centre lies within 3.5 dx of the origin (160 cells at any even n, reading R23)."""
    nx, ny, nz = (n, n, n) if np.isscalar(n) else n
    fs = [uniform_faces(-0.5, 0.5, m) for m in (nx, ny, nz)]
    gamma = 5.0 / 3.0
    spec = _spec("sedov_3d", 3, [nx, ny, nz], fs, [BC_TRANSMISSIVE] * 3, [BC_TRANSMISSIVE] * 3, gamma,
                 LIM_MINMOD, cfl=0.6, steps=100, seed=seed)
    dx = 1.0 / nx                              # reduced copies: radius in units of the x spacing
    cx, cy, cz = (centres(f) for f in fs)
    r2 = cz[:, None, None] ** 2 + cy[None, :, None] ** 2 + cx[None, None, :] ** 2
    inside = r2 < (3.5 * dx) ** 2
    ncell = int(inside.sum())
    W = np.zeros((5, nz, ny, nx))
    W[0] = 1.0 + 0.01 * noise(seed, (nz, ny, nx))
    W[4] = np.where(inside, (gamma - 1.0) * 1.0 / (ncell * (1.0 / nx) * (1.0 / ny) * (1.0 / nz)), 1e-5)
    spec["bomb_cells"] = ncell
    return spec, W


def rt_3d(n=512, seed=1004):
    """C4: 3-D Rayleigh-Taylor, n x n x n cells on [0,1]^2 x [0,2] (dz = 2 dx), periodic x/y,
    reflecting z, g = -0.1 z, 2 scalars, MC + HLLC, CFL 0.7, 50 steps (shape of PAPER.md Sect. 4.2,
    the paper's weak-scaling workload, App. B)."""
    nx, ny, nz = (n, n, n) if np.isscalar(n) else n
    fx = uniform_faces(0.0, 1.0, nx)
    fy = uniform_faces(0.0, 1.0, ny)
    fz = uniform_faces(0.0, 2.0, nz)
    g = -0.1
    spec = _spec("rt_3d", 3, [nx, ny, nz], [fx, fy, fz], [BC_PERIODIC, BC_PERIODIC, BC_REFLECTING],
                 [BC_PERIODIC, BC_PERIODIC, BC_REFLECTING], 1.4, LIM_MC, n_scalars=2,
                 gravity=GRAV_UNIFORM, g=(0.0, 0.0, g), cfl=0.7, steps=50, seed=seed)
    z = centres(fz)
    heavy = z > 1.0
    rho = np.where(heavy, 2.0, 1.0)
    p = 2.5 + g * rho * (z - 1.0)           # analytic piecewise hydrostatic column, P(1) = 2.5
    W = np.zeros((7, nz, ny, nx))
    W[0] = rho[:, None, None]
    W[3] = 0.01 * noise(seed, (nz, ny, nx)) * (np.abs(z - 1.0) < 0.05)[:, None, None]
    W[4] = p[:, None, None]
    W[5] = np.where(heavy, 1.0, 0.0)[:, None, None]
    W[6] = np.where(heavy, 0.0, 1.0)[:, None, None]
    return spec, W


def wedge_3d(n=(1024, 256, 256), seed=1005, n_scalars=4):
    """C5: spherical wedge, supernova-envelope-like (shape of PAPER.md Sect. 5.5): r in [1,100]
    log-spaced, theta in pi/2 +- 0.35, phi in +-0.35, gamma 4/3, rho ~ r^-2.5 with 1 % noise,
    hydrostatic P under point-mass gravity GM = 1, thermal bomb E = 10 in the first 4 radial
    cells (reading R24), 4 composition shells split at r = 3, 8, 25, reflecting r_min / theta /
    phi walls, transmissive r_max (R18), minmod + HLLC, CFL 0.6, 50 steps.  n_scalars = 5 adds a fifth shell
    boundary at r = 60 (the field count of the paper's supernova runs)."""
    nr, nt, nph = n
    fr = log_faces(1.0, 100.0, nr)
    ft = uniform_faces(math.pi / 2 - 0.35, math.pi / 2 + 0.35, nt)
    fph = uniform_faces(-0.35, 0.35, nph)
    gamma = 4.0 / 3.0
    spec = _spec("wedge_3d", 3, [nr, nt, nph], [fr, ft, fph], [BC_REFLECTING, BC_WEDGE, BC_WEDGE],
                 [BC_TRANSMISSIVE, BC_WEDGE, BC_WEDGE], gamma, LIM_MINMOD, coords=SPHERICAL, n_scalars=n_scalars,
                 gravity=GRAV_POINT_MASS, GM=1.0, cfl=0.6, steps=50, seed=seed)
    r = centres(fr)
    W = np.zeros((5 + n_scalars, nph, nt, nr))
    W[0] = (r ** -2.5)[None, None, :] * (1.0 + 0.01 * noise(seed, (nph, nt, nr)))
    p = r ** -3.5 / 3.5
    nb = min(4, nr)
    omega = (fph[-1] - fph[0]) * (math.cos(ft[0]) - math.cos(ft[-1]))
    v4 = (fr[nb] ** 3 - fr[0] ** 3) / 3.0 * omega
    p[:nb] += (gamma - 1.0) * 10.0 / v4
    W[4] = p[None, None, :]
    edges = [0.0, 3.0, 8.0, 25.0, 60.0][:n_scalars] + [np.inf]
    for s in range(n_scalars):
        W[5 + s] = ((r >= edges[s]) & (r < edges[s + 1])).astype(np.float64)[None, None, :]
    return spec, W


def sedov_wedge_3d(n=256, t_end=0.08):
    """SURVEY 8(f) rank 3, the paper's own spherical workload (Sect. 4.3): off-centre Sedov
    blast in a spherical wedge r in [0.1, 1.3], theta and phi in [pi/4, 3pi/4], 256^3 zones, rho0 = 1, P0 = 0.01,
    E1 = 1 at (r0, theta0, phi0) = (0.7, pi/2, pi/2), transmissive faces, gamma 5/3, run to t = 0.08.  The paper
    does not say how E1 is deposited, nor limiter / solver / CFL: here it is thermal energy spread uniformly (per
    volume) over the cells whose centre lies within 3.5 radial cell widths of the blast point, with minmod + HLLC
    at CFL 0.6 like the Cartesian Sedov configuration.  No noise: the setup is deterministic."""
    nr, nt, nph = (n, n, n) if np.isscalar(n) else n
    fr = uniform_faces(0.1, 1.3, nr)
    ft = uniform_faces(math.pi / 4, 3 * math.pi / 4, nt)
    fph = uniform_faces(math.pi / 4, 3 * math.pi / 4, nph)
    gamma = 5.0 / 3.0
    spec = _spec("sedov_wedge_3d", 3, [nr, nt, nph], [fr, ft, fph], [BC_TRANSMISSIVE] * 3, [BC_TRANSMISSIVE] * 3, gamma,
                 LIM_MINMOD, coords=SPHERICAL, cfl=0.6, steps=None, t_end=t_end, seed=0)
    r, th, ph = centres(fr), centres(ft), centres(fph)
    R, TH, PH = r[None, None, :], th[None, :, None], ph[:, None, None]
    r0, th0, ph0 = 0.7, math.pi / 2, math.pi / 2
    # Cartesian distance of the cell centres to the blast point
    x, y, z = R * np.sin(TH) * np.cos(PH), R * np.sin(TH) * np.sin(PH), R * np.cos(TH) + 0.0 * PH
    x0, y0, z0 = r0 * math.sin(th0) * math.cos(ph0), r0 * math.sin(th0) * math.sin(ph0), r0 * math.cos(th0)
    hot = (x - x0) ** 2 + (y - y0) ** 2 + (z - z0) ** 2 < (3.5 * (fr[1] - fr[0])) ** 2
    dV = ((fr[1:] ** 3 - fr[:-1] ** 3) / 3.0)[None, None, :] * (np.cos(ft[:-1]) - np.cos(ft[1:]))[None, :, None] \
        * (fph[1:] - fph[:-1])[:, None, None]
    W = np.zeros((5, nph, nt, nr))
    W[0] = 1.0
    W[4] = 0.01
    W[4][hot] = (gamma - 1.0) * 1.0 / float(np.sum(dV[hot]))
    return spec, W


def wedge_3d_rad(n=(1024, 256, 256), seed=1005):
    """the C5 wedge with the paper's production EOS for stellar explosions, an ideal gas in
    equilibrium with radiation (Eq. 6-7, used for the supernova runs, L377).  Same primitive
    fields (rho, u, P, f) as wedge_3d; gas gamma = 5/3, k_b/mu = 1, a_r = 30 in code units: P_r/P_g is 0.02-0.15 in the
    envelope (gas dominated, both terms matter) and about 16 in the bomb (radiation dominated)."""
    spec, W = wedge_3d(n, seed)
    spec = dict(spec, name="wedge_3d_rad", gamma=5.0 / 3.0, eos=EOS_GAS_RADIATION, eos_R=1.0, eos_ar=30.0)
    return spec, W


def wedge_3d_sn(n=(1024, 256, 256), seed=1005):
    """The setup of the paper's second weak-scaling run ("3-D spherical, gas + radiation EOS, 5 passive
    scalars, point-mass gravity"): wedge_3d_rad with five composition shells (nvar 10)."""
    spec, W = wedge_3d(n, seed, n_scalars=5)
    spec = dict(spec, name="wedge_3d_sn", gamma=5.0 / 3.0, eos=EOS_GAS_RADIATION, eos_R=1.0, eos_ar=30.0)
    return spec, W


def wedge_3d_emon(n=(1024, 256, 256), seed=1007, n_scalars=4):
    """SURVEY 8(f) rank 2 in the geometry the paper uses it for ("highly supersonic" supernova ejecta):
    the C5 wedge (same grid, density, pressure without the bomb, four composition shells, point-mass gravity) as a cold
    radial outflow u_r = 500 (Mach 800 at r = 1, 8000 at r = 100) with seeded velocity noise of 0.3 c_s in all three
    components (subsonic in the comoving frame), transmissive radial faces, monitoring with the paper's epsilon = 1e-6.
    e / e_k = 6.8e-6 / r: alpha = 1 inside r ~ 7, the blended branch of Eq. 12 out to r ~ 68, alpha = 0 (internal energy
    from Eq. 10 alone) beyond.  (A homologous outflow u_r ~ r at this Mach number breaks the scheme in its first step
    with or without monitoring: the Hancock predictor forms its pressures from the total energy, R29.)"""
    spec, W = wedge_3d(n, seed, n_scalars=n_scalars)
    nr, nt, nph = n
    spec = dict(spec, name="wedge_3d_emon", emon_eps=1e-6)
    spec["bc_lo"] = [BC_TRANSMISSIVE, BC_WEDGE, BC_WEDGE]
    r = centres(spec["faces"][0])
    W[4] = (r ** -3.5 / 3.5)[None, None, :] + 0.0 * W[4]          # no bomb
    cs = np.sqrt(4.0 / 3.0 * (r ** -3.5 / 3.5) / r ** -2.5)
    W[1] = 500.0 + 0.3 * cs[None, None, :] * noise(seed + 1, (nph, nt, nr))
    W[2] = 0.3 * cs[None, None, :] * noise(seed + 2, (nph, nt, nr))
    W[3] = 0.3 * cs[None, None, :] * noise(seed + 3, (nph, nt, nr))
    return spec, W


def wedge_3d_sn_emon(n=(1024, 256, 256), seed=1007):
    """Everything the paper's supernova runs switch on at once: the cold supersonic outflow of
    wedge_3d_emon with five composition shells (nvar 10), the gas + radiation EOS (gas gamma 5/3, k_b/mu = 1, a_r = 30 as in
    wedge_3d_rad: the same rho and P give P_r / P_g of 0.02-0.15), point-mass gravity and the monitoring of the internal energy."""
    spec, W = wedge_3d_emon(n, seed, n_scalars=5)
    spec = dict(spec, name="wedge_3d_sn_emon", gamma=5.0 / 3.0, eos=EOS_GAS_RADIATION, eos_R=1.0, eos_ar=30.0)
    return spec, W


def wedge_3d_selfgrav(n=(1024, 256, 256), seed=1005):
    """the C5 wedge with the self-gravity of its envelope (Eq. 4) on top of the
    central mass: G M_c = 1 as in wedge_3d, G = 0.004, so that the spherically averaged envelope (mass 8 pi (sqrt(r) - 1)
    inside r for rho = r^-2.5) adds G M_env ~ 0.9 at r = 100, comparable to the central mass.  Same primitive
    fields as wedge_3d (its pressure balances the central mass only: the envelope starts to contract slowly)."""
    spec, W = wedge_3d(n, seed)
    spec = dict(spec, name="wedge_3d_selfgrav", gravity=GRAV_SELF, G=0.004)
    return spec, W


def cold_stream_3d(n=256, seed=1006):
    """a workload for the monitoring of the internal energy in highly supersonic regions (PAPER.md
    Eq. 10-12): a cold stream, Mach ~ 2800, crossing a periodic unit box with 20 % density and 10 % pressure
    structure and 0.01 % seeded velocity noise (0.3, subsonic in the stream frame); e / e_k ~ 4e-7, so that with the paper's epsilon = 1e-6 the cells sit on the
    blended branch of Eq. 12 (alpha ~ 0.1-0.2).  gamma = 1.4, MC + HLLC, CFL 0.6, 50 steps."""
    nx, ny, nz = (n, n, n) if np.isscalar(n) else n
    fs = [uniform_faces(0.0, 1.0, m) for m in (nx, ny, nz)]
    spec = _spec("cold_stream_3d", 3, [nx, ny, nz], fs, [BC_PERIODIC] * 3, [BC_PERIODIC] * 3, 1.4, LIM_MC, cfl=0.6, steps=50,
                 seed=seed, emon_eps=1e-6)
    x, y, z = centres(fs[0])[None, None, :], centres(fs[1])[None, :, None], centres(fs[2])[:, None, None]
    W = np.empty((5, nz, ny, nx))
    W[0] = 1.0 + 0.2 * np.sin(2 * math.pi * x) * np.cos(2 * math.pi * y) + 0.0 * z
    W[1] = 3000.0 * (1.0 + 1e-4 * noise(seed, (nz, ny, nx)))
    W[2] = -2000.0
    W[3] = 1000.0
    W[4] = 1.0 + 0.1 * np.cos(2 * math.pi * z) * np.sin(2 * math.pi * x) + 0.0 * y
    return spec, W


CONFIGS = {"sod_1d": sod_1d, "kh_2d": kh_2d, "sedov_3d": sedov_3d, "rt_3d": rt_3d, "wedge_3d": wedge_3d}


def smooth_periodic(ndim, n, seed=7, n_scalars=1, coords=CARTESIAN, limiter=LIM_VANLEER, riemann=RIEMANN_HLLC,
                    gamma=1.4, amp=0.2):
    """Random smooth periodic state (a few low Fourier modes per field) for invariant tests."""
    rng = np.random.default_rng(seed)
    n = list(n)
    faces = [uniform_faces(0.0, 1.0, m) for m in n]
    spec = _spec("smooth_periodic", ndim, n, faces, [BC_PERIODIC] * ndim, [BC_PERIODIC] * ndim, gamma, limiter,
                 riemann=riemann, coords=coords, n_scalars=n_scalars, cfl=0.4, seed=seed)
    n3 = n + [1] * (3 - ndim)
    grids = np.meshgrid(*[centres(f) for f in faces][::-1], indexing="ij") if ndim > 1 else [centres(faces[0])]
    grids = grids[::-1]  # grids[d] varies along direction d; arrays are indexed [.., j, i]

    def field(mean, a):
        out = np.full(n3[::-1][3 - ndim:], mean, dtype=np.float64)
        for _ in range(3):
            ph = rng.uniform(0, 2 * math.pi)
            kv = rng.integers(0, 3, size=ndim)
            if not kv.any():
                kv[0] = 1
            arg = sum(2 * math.pi * kv[d] * grids[d] for d in range(ndim)) + ph
            out = out + a * rng.uniform(0.3, 1.0) * np.sin(arg)
        return out

    nvar = 2 + ndim + n_scalars
    W = np.empty((nvar,) + tuple(n3[::-1]))
    W[0] = field(1.0, amp / 3).reshape(n3[::-1])
    for d in range(ndim):
        W[1 + d] = field(rng.uniform(-0.3, 0.3), amp).reshape(n3[::-1])
    W[1 + ndim] = field(1.0, amp / 3).reshape(n3[::-1])
    for s in range(n_scalars):
        W[2 + ndim + s] = field(0.5, amp / 2).reshape(n3[::-1])
    return spec, W

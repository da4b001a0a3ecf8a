"""Pins of the CPU oracle against things other than itself (CPU only, `-m "not gpu"`).

P1  Sod tube vs the exact Riemann solution (tests/exact_riemann.py) and Toro's printed star state
P2  smooth advection / isentropic vortex: measured order of accuracy (1st order NONE, ~2nd MUSCL-Hancock)
P3  uniform state preserved (bitwise Cartesian periodic; <=1e-14 spherical at rest)
P4  conservation of mass, momentum, energy, scalars in a periodic box to round-off
P5  F(U,U) = analytic flux; stationary contact exactly preserved by HLLC and smeared by HLL
P6  mirror symmetry; Sod along x, y, z inside a 3-D grid equals the 1-D run
P7  angular momentum sum(rho u_phi r_c s_c dV) conserved (Eq. 14 identity)
P8  spherical Sedov: shock radius vs Eq. 25; 3-D wedge equals the 1-D run
P9  uniform free fall exact with the time-centred gravity source
P10 hydrostatic column stays (nearly) at rest; closed reflecting box conserves mass with gravity (R25)
P11 brute force: naive per-cell evaluation == whole-array passes on tiny grids, every BC / geometry
plus closed forms of the limiters and geometry.
"""
import math
import os

import numpy as np
import pytest

from paper_2503_04428_b200 import workloads as wl
from tests import exact_riemann
from tests.helpers import fsum, read_golden, run_steps, run_to_time

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def make(ox, spec, W):
    o = ox.Oracle(spec)
    o.set_state(W, ox.PRIMITIVE)
    return o


# ------------------------------------------------------------------------------------------ P1
def sod_error(ox, n, limiter, riemann):
    spec, W = wl.sod_1d(n)
    spec["limiter"], spec["riemann"] = limiter, riemann
    o = make(ox, spec, W)
    run_to_time(o, 0.8, 0.2)
    P = o.get_state(ox.PRIMITIVE)
    x = wl.centres(spec["faces"][0])
    rho, u, p = exact_riemann.sample((1.0, 0.0, 1.0), (0.125, 0.0, 0.1), 1.4, (x - 0.5) / 0.2)
    dx = 1.0 / n
    return (np.sum(np.abs(P[0, 0, 0] - rho)) * dx, np.sum(np.abs(P[1, 0, 0] - u)) * dx,
            np.sum(np.abs(P[2, 0, 0] - p)) * dx), P


def test_exact_solver_matches_printed_star_state():
    g = read_golden(os.path.join(GOLDEN, "sod_star_state.txt"))
    ps, us = exact_riemann.star_state((1.0, 0.0, 1.0), (0.125, 0.0, 0.1), 1.4)
    assert abs(ps - g["p_star"]) < 1e-5 and abs(us - g["u_star"]) < 1e-5
    rho, _, _ = exact_riemann.sample((1.0, 0.0, 1.0), (0.125, 0.0, 0.1), 1.4, [us - 1e-3, us + 1e-3])
    assert abs(rho[0] - g["rho_star_left"]) < 1e-5 and abs(rho[1] - g["rho_star_right"]) < 1e-5


@pytest.mark.parametrize("riemann", [0, 1])
@pytest.mark.parametrize("limiter", [0, 1, 2, 3, 4])
def test_p1_sod_converges_to_exact(oxlib, limiter, riemann):
    ox = oxlib
    errs = [sod_error(ox, n, limiter, riemann)[0] for n in (100, 200, 400, 800)]
    rho_err = [e[0] for e in errs]
    for a, b in zip(rho_err, rho_err[1:]):
        assert b < a, rho_err
    order = math.log(rho_err[0] / rho_err[-1]) / math.log(8.0)
    if limiter == 0:
        assert 0.45 < order < 0.95, order    # first-order scheme on a discontinuous solution
        assert rho_err[0] < 2.5e-2
    else:
        assert 0.7 < order < 1.2, order      # MUSCL-Hancock on a discontinuous solution
        assert rho_err[0] < 1.0e-2
    for e in errs[-1]:
        assert e < 5e-3


def test_p1_sod_star_plateau_matches_printed_values(oxlib):
    g = read_golden(os.path.join(GOLDEN, "sod_star_state.txt"))
    _, P = sod_error(oxlib, 1000, 1, 1)
    x = (np.arange(1000) + 0.5) / 1000
    left_star = (x > 0.56) & (x < 0.66)      # between rarefaction tail (0.486) and contact (0.685)
    right_star = (x > 0.72) & (x < 0.82)     # between contact and shock (0.850)
    assert np.max(np.abs(P[2, 0, 0][left_star] - g["p_star"])) < 2e-3
    assert np.max(np.abs(P[1, 0, 0][left_star] - g["u_star"])) < 2e-3
    assert np.max(np.abs(P[0, 0, 0][left_star] - g["rho_star_left"])) < 2e-3
    assert np.max(np.abs(P[0, 0, 0][right_star] - g["rho_star_right"])) < 2e-3


# ------------------------------------------------------------------------------------------ P2
def advect_error(ox, ndim, n, limiter, cfl, riemann=1, t_end=1.0):
    faces = [wl.uniform_faces(0.0, 1.0, n) for _ in range(ndim)]
    spec = wl._spec("advect", ndim, [n] * ndim, faces, [0] * ndim, [0] * ndim, 1.4, limiter, riemann=riemann)
    c = wl.centres(faces[0])
    shape = [1, 1, 1]
    s = 0.0
    for d in range(ndim):
        sh = [1, 1, 1]
        sh[2 - d] = n
        s = s + c.reshape(sh)
        shape[2 - d] = n
    W = np.empty((2 + ndim,) + tuple(shape))
    W[0] = 1.0 + 0.2 * np.sin(2 * math.pi * s)
    for d in range(ndim):
        W[1 + d] = 1.0
    W[1 + ndim] = 1.0
    o = make(ox, spec, W)
    run_to_time(o, cfl, t_end)
    P = o.get_state(ox.PRIMITIVE)
    exact = 1.0 + 0.2 * np.sin(2 * math.pi * (s - ndim * t_end))     # profile carried by u = (1,..,1)
    return float(np.mean(np.abs(P[0] - exact)))


@pytest.mark.parametrize("ndim,sizes,cfl", [(1, (32, 64, 128), 0.8), (2, (16, 32, 64), 0.8), (3, (8, 16, 32), 0.6)])
def test_p2_advection_order(oxlib, ndim, sizes, cfl):
    # first order (limiter NONE): short run so that the donor-cell damping stays in the asymptotic regime
    e1 = [advect_error(oxlib, ndim, n, 0, cfl, t_end=0.05) for n in sizes[1:]]
    assert 0.75 < math.log2(e1[0] / e1[1]) < 1.25, e1
    # MUSCL-Hancock: second order away from the (clipped) extrema; the 3-D sizes the CPU suite can
    # afford (16 -> 32 cells per wavelength) are still pre-asymptotic, hence the lower bar there
    bars = ((2, 1.8), (4, 1.8), (3, 1.7), (1, 1.3)) if ndim < 3 else ((2, 1.4), (4, 1.4), (1, 1.1))
    for lim, lo in bars:
        e = [advect_error(oxlib, ndim, n, lim, cfl) for n in sizes[1:]]
        order = math.log2(e[0] / e[1])
        assert lo < order < 3.2, (lim, e, order)


def vortex_error(ox, n, limiter, riemann):
    """2-D isentropic vortex (exact steady solution advected by a uniform flow), periodic box."""
    L = 10.0
    faces = [wl.uniform_faces(-L / 2, L / 2, n)] * 2
    gamma = 1.4
    spec = wl._spec("vortex", 2, [n, n], faces, [0, 0], [0, 0], gamma, limiter, riemann=riemann)
    c = wl.centres(faces[0])
    X, Y = np.meshgrid(c, c, indexing="xy")      # arrays indexed [j, i]
    beta = 5.0
    r2 = X * X + Y * Y
    dT = -(gamma - 1.0) * beta ** 2 / (8 * gamma * math.pi ** 2) * np.exp(1.0 - r2)
    W = np.empty((4, 1, n, n))
    W[0, 0] = (1.0 + dT) ** (1.0 / (gamma - 1.0))
    W[1, 0] = 1.0 - beta / (2 * math.pi) * np.exp(0.5 * (1.0 - r2)) * Y
    W[2, 0] = 1.0 + beta / (2 * math.pi) * np.exp(0.5 * (1.0 - r2)) * X
    W[3, 0] = (1.0 + dT) ** (gamma / (gamma - 1.0))
    o = make(ox, spec, W)
    run_to_time(o, 0.8, L)                       # one period: the vortex returns to its start
    P = o.get_state(ox.PRIMITIVE)
    return [float(np.mean(np.abs(P[v] - W[v]))) for v in range(4)]


@pytest.mark.parametrize("riemann", [0, 1])
def test_p2_isentropic_vortex_second_order(oxlib, riemann):
    e32 = vortex_error(oxlib, 32, 2, riemann)
    e64 = vortex_error(oxlib, 64, 2, riemann)
    for v in range(4):   # density, both momenta (cross terms rho u_x u_y), pressure
        order = math.log2(e32[v] / e64[v])
        assert 1.6 < order < 3.2, (v, e32, e64)


# ------------------------------------------------------------------------------------------ P3
@pytest.mark.parametrize("ndim", [1, 2, 3])
def test_p3_uniform_state_cartesian_bitwise(oxlib, ndim):
    ox = oxlib
    n = [12, 10, 8][:ndim]
    faces = [wl.uniform_faces(0.0, 1.0 + d, m) for d, m in enumerate(n)]
    for limiter in (0, 1, 4):
        for riemann in (0, 1):
            spec = wl._spec("uni", ndim, n, faces, [0] * ndim, [0] * ndim, 1.4, limiter, riemann=riemann, n_scalars=2)
            W = np.empty((4 + ndim,) + tuple((n + [1, 1])[:3][::-1]))
            vals = [1.37, 0.31, -0.47, 0.22][: 1 + ndim] + [0.83, 0.25, 0.75]
            for v, x in enumerate(vals):
                W[v] = x
            o = make(ox, spec, W)
            U0 = o.get_state()
            run_steps(o, 0.5, 3)
            assert np.array_equal(o.get_state(), U0)


@pytest.mark.parametrize("ndim", [1, 2, 3])
def test_p3_uniform_rest_state_spherical(oxlib, ndim):
    ox = oxlib
    n = [16, 8, 6][:ndim]
    faces = [wl.log_faces(0.5, 4.0, n[0])]
    if ndim >= 2:
        faces.append(wl.uniform_faces(0.6, 2.2, n[1]))
    if ndim >= 3:
        faces.append(wl.uniform_faces(-0.4, 0.7, n[2]))
    bc = [ox.BC_REFLECTING, ox.BC_WEDGE, ox.BC_WEDGE][:ndim]
    for limiter in (0, 1, 2):
        spec = wl._spec("uni_sph", ndim, n, faces, bc, bc, 5.0 / 3.0, limiter, coords=ox.SPHERICAL, n_scalars=1)
        W = np.zeros((3 + ndim,) + tuple((n + [1, 1])[:3][::-1]))
        W[0], W[1 + ndim], W[2 + ndim] = 1.3, 0.7, 0.4
        o = make(ox, spec, W)
        U0 = o.get_state()
        run_steps(o, 0.5, 3)
        U1 = o.get_state()
        scale = np.max(np.abs(U0))
        assert np.max(np.abs(U1 - U0)) <= 3e-14 * scale


# ------------------------------------------------------------------------------------------ P4
@pytest.mark.parametrize("ndim,n", [(1, [64]), (2, [24, 20]), (3, [12, 10, 8])])
@pytest.mark.parametrize("riemann", [0, 1])
def test_p4_conservation_periodic(oxlib, ndim, n, riemann):
    ox = oxlib
    spec, W = wl.smooth_periodic(ndim, n, seed=11 + ndim, n_scalars=2, limiter=ox.LIM_MC, riemann=riemann)
    o = make(ox, spec, W)
    U0 = o.get_state()
    run_steps(o, 0.5, 100 if ndim < 3 else 40)
    U1 = o.get_state()
    for v in range(U0.shape[0]):
        s0, s1 = fsum(U0[v]), fsum(U1[v])
        scale = fsum(np.abs(U0[v]))
        assert abs(s1 - s0) <= 1e-13 * scale, (v, s0, s1)
    assert np.max(np.abs(U1 - U0)) > 1e-3     # the state did evolve


# ------------------------------------------------------------------------------------------ P5
def random_state(rng, ndim, ns):
    W = np.concatenate([[rng.uniform(0.2, 3.0)], rng.uniform(-2, 2, ndim), [rng.uniform(0.1, 4.0)], rng.uniform(0, 1, ns)])
    rho, u, p, f = W[0], W[1:1 + ndim], W[1 + ndim], W[2 + ndim:]
    gamma = 1.4
    return np.concatenate([[rho], rho * u, [p / (gamma - 1) + 0.5 * rho * np.dot(u, u)], rho * f]), W


@pytest.mark.parametrize("ndim", [1, 2, 3])
def test_p5_consistency_and_closed_form_flux(oxlib, ndim):
    ox = oxlib
    rng = np.random.default_rng(5)
    gamma = 1.4
    for _ in range(50):
        U, W = random_state(rng, ndim, 2)
        for d in range(ndim):
            rho, u, p, f = W[0], W[1:1 + ndim], W[1 + ndim], W[2 + ndim:]
            E = U[1 + ndim]
            mom = rho * u * u[d]
            mom[d] += p
            Fexp = np.concatenate([[rho * u[d]], mom, [(E + p) * u[d]], rho * f * u[d]])   # Eq. 1, retyped
            Fphys = ox.physical_flux(gamma, ndim, 2, d, U)
            assert np.allclose(Fphys, Fexp, rtol=1e-14, atol=1e-14)
            for riemann in (0, 1):
                F = ox.riemann_flux(riemann, gamma, ndim, 2, d, U, U)
                assert np.allclose(F, Fexp, rtol=2e-14, atol=2e-14), (riemann, d)


def test_p5_supersonic_upwinding(oxlib):
    ox = oxlib
    gamma = 1.4
    WL = np.array([1.0, 5.0, 0.3, 1.0, 0.2])
    WR = np.array([0.5, 4.0, -0.2, 0.4, 0.9])   # both supersonic to the right (c ~ 1.2)

    def cons(W):
        return np.array([W[0], W[0] * W[1], W[0] * W[2], W[3] / (gamma - 1) + 0.5 * W[0] * (W[1] ** 2 + W[2] ** 2), W[0] * W[4]])
    for riemann in (0, 1):
        F = ox.riemann_flux(riemann, gamma, 2, 1, 0, cons(WL), cons(WR))
        assert np.array_equal(F, ox.physical_flux(gamma, 2, 1, 0, cons(WL)))
        WLm, WRm = WL.copy(), WR.copy()
        WLm[1], WRm[1] = -4.0, -5.0
        F = ox.riemann_flux(riemann, gamma, 2, 1, 0, cons(WLm), cons(WRm))
        assert np.array_equal(F, ox.physical_flux(gamma, 2, 1, 0, cons(WRm)))


def test_p5_stationary_contact(oxlib):
    ox = oxlib
    n = 64
    fx = wl.uniform_faces(0.0, 1.0, n)
    W = np.zeros((4, 1, 1, n))
    W[0, 0, 0] = np.where(wl.centres(fx) < 0.5, 1.0, 0.125)
    W[2] = 1.0
    W[3, 0, 0] = np.where(wl.centres(fx) < 0.5, 1.0, 0.0)
    out = {}
    for riemann in (0, 1):
        spec = wl._spec("contact", 1, [n], [fx], [1], [1], 1.4, ox.LIM_MINMOD, riemann=riemann, n_scalars=1)
        o = make(ox, spec, W)
        run_steps(o, 0.8, 50)
        out[riemann] = o.get_state(ox.PRIMITIVE)
    assert np.array_equal(out[1], W)                             # HLLC: exactly sharp for all time
    assert np.sum(np.abs(out[0][0] - W[0])) / n > 1e-3           # HLL smears it
    assert np.max(np.abs(out[0][1])) < 1e-13 and np.max(np.abs(out[0][2] - 1.0)) < 1e-13


# ------------------------------------------------------------------------------------------ P6
def test_p6_sod_along_each_axis_equals_1d(oxlib):
    ox = oxlib
    n = 48
    fx = wl.uniform_faces(0.0, 1.0, n)
    ft = wl.uniform_faces(0.0, 0.25, 4)
    c = wl.centres(fx)
    rho = np.where(c < 0.5, 1.0, 0.125)
    p = np.where(c < 0.5, 1.0, 0.1)
    f = np.where(c < 0.5, 1.0, 0.0)
    results = []
    dts = None
    for axis in (0, 1, 2):
        nn = [4, 4, 4]
        nn[axis] = n
        faces = [ft, ft, ft]
        faces[axis] = fx
        spec = wl._spec("sod3", 3, nn, faces, [1, 1, 1], [1, 1, 1], 1.4, ox.LIM_VANLEER, n_scalars=1)
        sh = [1, 1, 1]
        sh[2 - axis] = n
        W = np.zeros((6,) + tuple(nn[::-1]))
        W[0] = rho.reshape(sh)
        W[4] = p.reshape(sh)
        W[5] = f.reshape(sh)
        o = make(ox, spec, W)
        if dts is None:
            dts = run_steps(o, 0.6, 25)
        else:
            for dt in dts:
                o.step(dt)
        U = o.get_state()
        line = np.moveaxis(U, 3 - axis, -1)[:, 1, 2, :]       # any transverse position
        assert np.max(np.abs(np.moveaxis(U, 3 - axis, -1) - line[:, None, None, :])) == 0.0
        order = [0, 1 + axis, 4, 5]                            # rho, normal momentum, E, scalar
        results.append(line[order])
        for d in range(3):
            if d != axis:
                assert np.max(np.abs(U[1 + d])) == 0.0
    spec1 = wl._spec("sod1", 1, [n], [fx], [1], [1], 1.4, ox.LIM_VANLEER, n_scalars=1)
    W1 = np.zeros((4, 1, 1, n))
    W1[0, 0, 0], W1[2, 0, 0], W1[3, 0, 0] = rho, p, f
    o1 = make(ox, spec1, W1)
    for dt in dts:
        o1.step(dt)
    U1 = o1.get_state()[:, 0, 0, :]
    for r in results:
        assert np.max(np.abs(r - U1)) <= 1e-14
    assert np.max(np.abs(results[0] - results[1])) <= 1e-15 and np.max(np.abs(results[0] - results[2])) <= 1e-15


def test_p6_mirror_symmetry_blast(oxlib):
    ox = oxlib
    n = 16
    f = wl.uniform_faces(-0.5, 0.5, n)
    spec = wl._spec("blast", 3, [n] * 3, [f] * 3, [1] * 3, [1] * 3, 5.0 / 3.0, ox.LIM_MINMOD)
    c = wl.centres(f)
    r2 = c[:, None, None] ** 2 + c[None, :, None] ** 2 + c[None, None, :] ** 2
    W = np.zeros((5, n, n, n))
    W[0] = 1.0
    W[4] = np.where(r2 < (2.5 / n) ** 2, 10.0, 0.1)
    o = make(ox, spec, W)
    run_steps(o, 0.6, 12)
    U = o.get_state()
    scale = np.max(np.abs(U), axis=(1, 2, 3), keepdims=True)
    for axis, mom in ((3, 1), (2, 2), (1, 3)):
        Um = np.flip(U, axis=axis).copy()
        Um[mom] *= -1.0
        assert np.max(np.abs(Um - U) / scale) <= 1e-13
    # permutation symmetry x <-> y
    Ut = np.swapaxes(U, 2, 3).copy()
    Ut[[1, 2]] = Ut[[2, 1]]
    assert np.max(np.abs(Ut - U) / scale) <= 1e-13
    assert np.max(np.abs(U[1])) > 1e-2


# ------------------------------------------------------------------------------------------ P7
def test_p7_angular_momentum(oxlib):
    ox = oxlib
    n = [20, 12, 16]
    fr = wl.uniform_faces(1.0, 2.0, n[0])
    ft = wl.uniform_faces(0.9, 2.1, n[1])
    fp = wl.uniform_faces(0.0, 1.6, n[2])
    spec = wl._spec("angmom", 3, n, [fr, ft, fp], [2, 3, 0], [2, 3, 0], 1.4, ox.LIM_VANLEER, coords=ox.SPHERICAL, n_scalars=0)
    r, t, p = wl.centres(fr), wl.centres(ft), wl.centres(fp)
    R, T, PH = r[None, None, :], t[None, :, None], p[:, None, None]
    bump = np.exp(-((R - 1.5) / 0.12) ** 2 - ((T - 1.5) / 0.15) ** 2)       # vanishes (<1e-7) at the r, theta walls
    bump = np.where(bump < 1e-6, 0.0, bump) * (1.0 + 0.3 * np.sin(2 * math.pi * PH / 1.6))
    W = np.zeros((5, n[2], n[1], n[0]))
    W[0] = 1.0 + 0.5 * bump
    W[1] = 0.2 * bump
    W[2] = -0.15 * bump
    W[3] = 0.6 * bump
    W[4] = 1.0 + 0.3 * bump
    o = make(ox, spec, W)

    def angmom():
        U = o.get_state()
        tot = 0.0
        terms = []
        for k in range(n[2]):
            for j in range(n[1]):
                for i in range(n[0]):
                    dV, _, xc = o.cell_geometry(i, j, k)
                    sc = 0.5 * (math.sin(ft[j]) + math.sin(ft[j + 1]))
                    terms.append(U[3, k, j, i] * xc[0] * sc * dV)
        return math.fsum(terms), math.fsum(abs(x) for x in terms)
    L0, scale = angmom()
    run_steps(o, 0.5, 6)
    L1, _ = angmom()
    assert scale > 1e-4
    assert abs(L1 - L0) <= 1e-13 * scale, (L0, L1, scale)
    U = o.get_state()
    assert np.max(np.abs(U[3] - W[0] * W[3])) > 1e-3


# ------------------------------------------------------------------------------------------ P8
def sedov_1d_spec(ox, n, gamma):
    fr = wl.uniform_faces(0.0, 1.0, n)
    spec = wl._spec("sedov1", 1, [n], [fr], [ox.BC_REFLECTING], [ox.BC_TRANSMISSIVE], gamma, ox.LIM_MINMOD, coords=ox.SPHERICAL)
    W = np.zeros((3, 1, 1, n))
    W[0] = 1.0
    W[2] = 1e-6
    nb = 2
    vol = 4.0 * math.pi / 3.0 * fr[nb] ** 3                 # inactive angles default to the full sphere
    W[2, 0, 0, :nb] = (gamma - 1.0) * 1.0 / vol
    return spec, W, fr


@pytest.mark.parametrize("gamma,key", [(1.4, "gamma_1_4"), (5.0 / 3.0, "gamma_5_3")])
def test_p8_spherical_sedov_shock_radius(oxlib, gamma, key):
    ox = oxlib
    xi0 = read_golden(os.path.join(GOLDEN, "sedov_similarity.txt"))[key]
    spec, W, fr = sedov_1d_spec(ox, 400, gamma)
    o = make(ox, spec, W)
    t_end = 0.3
    run_to_time(o, 0.6, t_end)
    P = o.get_state(ox.PRIMITIVE)
    r = wl.centres(fr)
    r_shock = r[np.argmax(P[0, 0, 0])]
    expected = xi0 * (1.0 * t_end ** 2 / 1.0) ** 0.2
    assert abs(r_shock - expected) / expected < 0.04, (r_shock, expected)
    # strong-shock density jump (gamma+1)/(gamma-1), smeared by the scheme
    assert 0.6 * (gamma + 1) / (gamma - 1) < P[0].max() < 1.02 * (gamma + 1) / (gamma - 1)
    # total energy conserved in the closed sphere until the shock reaches the outer boundary
    U = o.get_state()
    vols = 4.0 * math.pi / 3.0 * (fr[1:] ** 3 - fr[:-1] ** 3)
    e_tot = fsum(U[2, 0, 0] * vols)
    e0 = 1.0 + 1e-6 / (gamma - 1) * 4 * math.pi / 3 * (1 - fr[2] ** 3)
    assert abs(e_tot - e0) < 1e-11


@pytest.mark.parametrize("ndim", [2, 3])
def test_p8_wedge_equals_1d_spherical(oxlib, ndim):
    ox = oxlib
    n = 48
    gamma = 1.4
    fr = wl.log_faces(0.2, 2.0, n)
    r = wl.centres(fr)
    rho = 1.0 + 0.5 * np.exp(-((r - 0.9) / 0.2) ** 2)
    ur = 0.4 * np.sin(3.0 * r)
    p = 1.0 + 2.0 * np.exp(-((r - 0.6) / 0.15) ** 2)
    f = 0.5 + 0.5 * np.tanh((r - 1.0) / 0.1)
    nn = [n, 4, 4][:ndim]
    faces = [fr, wl.uniform_faces(1.1, 1.5, 4), wl.uniform_faces(-0.2, 0.3, 4)][:ndim]
    bc_lo = [ox.BC_REFLECTING, ox.BC_WEDGE, ox.BC_WEDGE][:ndim]
    bc_hi = [ox.BC_TRANSMISSIVE, ox.BC_WEDGE, ox.BC_WEDGE][:ndim]
    kw = dict(coords=ox.SPHERICAL, n_scalars=1, gravity=ox.GRAV_POINT_MASS, GM=0.7)
    spec = wl._spec("wedge_small", ndim, nn, faces, bc_lo, bc_hi, gamma, ox.LIM_VANLEER, **kw)
    shape = tuple((nn + [1, 1])[:3][::-1])
    W = np.zeros((3 + ndim,) + shape)
    W[0], W[1], W[1 + ndim], W[2 + ndim] = rho, ur, p, f
    o = make(ox, spec, W)
    dts = run_steps(o, 0.5, 20)
    U = o.get_state()
    spec1 = wl._spec("r_only", 1, [n], [fr], bc_lo[:1], bc_hi[:1], gamma, ox.LIM_VANLEER, **kw)
    # the 1-D run sees the same solid-angle-independent problem: give it the wedge's angular extents
    spec1["lo"][1], spec1["hi"][1] = 1.1, 1.5
    spec1["lo"][2], spec1["hi"][2] = -0.2, 0.3
    W1 = np.zeros((4, 1, 1, n))
    W1[0, 0, 0], W1[1, 0, 0], W1[2, 0, 0], W1[3, 0, 0] = rho, ur, p, f
    o1 = make(ox, spec1, W1)
    for dt in dts:
        o1.step(dt)
    U1 = o1.get_state()[:, 0, 0, :]
    pick = [0, 1, 1 + ndim, 2 + ndim]
    for k in range(shape[0]):
        for j in range(shape[1]):
            for a, v in enumerate(pick):
                assert np.max(np.abs(U[v, k, j] - U1[a])) <= 1e-12 * np.max(np.abs(U1[a]))
    for d in range(1, ndim):
        assert np.max(np.abs(U[1 + d])) <= 1e-12
    assert np.max(np.abs(U1[1] - rho * ur)) > 1e-2


# ------------------------------------------------------------------------------------------ P9
@pytest.mark.parametrize("ndim", [1, 2, 3])
def test_p9_uniform_free_fall(oxlib, ndim):
    ox = oxlib
    n = [8, 6, 4][:ndim]
    faces = [wl.uniform_faces(0.0, 1.0, m) for m in n]
    g = [0.3, -0.7, 0.45][:ndim] + [0.0] * (3 - ndim)
    spec = wl._spec("fall", ndim, n, faces, [0] * ndim, [0] * ndim, 1.4, ox.LIM_MC, gravity=ox.GRAV_UNIFORM, g=g, n_scalars=1)
    shape = tuple((n + [1, 1])[:3][::-1])
    W = np.zeros((3 + ndim,) + shape)
    u0 = [0.2, -0.1, 0.05][:ndim]
    W[0] = 1.7
    for d in range(ndim):
        W[1 + d] = u0[d]
    W[1 + ndim] = 0.9
    W[2 + ndim] = 0.3
    o = make(ox, spec, W)
    dts = run_steps(o, 0.5, 30)
    t = sum(dts)
    P = o.get_state(ox.PRIMITIVE)
    for d in range(ndim):
        assert np.max(np.abs(P[1 + d] - (u0[d] + g[d] * t))) <= 1e-13
    assert np.max(np.abs(P[0] - 1.7)) == 0.0
    assert np.max(np.abs(P[1 + ndim] - 0.9)) <= 1e-13
    assert np.max(np.abs(P[2 + ndim] - 0.3)) <= 1e-15


# ------------------------------------------------------------------------------------------ P10
def test_p10_hydrostatic_column_and_closed_box_mass(oxlib):
    ox = oxlib
    spec, W = wl.rt_3d(16, seed=3)
    W[3] = 0.0                                   # no velocity perturbation
    o = make(ox, spec, W)
    U0 = o.get_state()
    run_steps(o, 0.7, 30)
    P = o.get_state(ox.PRIMITIVE)
    assert np.max(np.abs(P[3])) < 5e-3           # residual O(dz^2) at the density jump, not growing wildly
    assert np.max(np.abs(P[1])) == 0.0 and np.max(np.abs(P[2])) == 0.0
    U1 = o.get_state()
    # reflecting z walls with mirrored gravity (R25): no mass, scalar or horizontal-momentum leak
    for v in (0, 5, 6):
        assert abs(fsum(U1[v]) - fsum(U0[v])) <= 1e-13 * fsum(np.abs(U0[v]))


def test_p10_rt_growth_is_physical(oxlib):
    """Heavy fluid on top is unstable under g pointing down and stable when g points up (sign of gravity, R12)."""
    ox = oxlib
    out = []
    for g in (-0.5, 0.5):
        spec, W = wl.rt_3d(16, seed=3)
        spec["g"] = [0.0, 0.0, g]
        z = wl.centres(spec["faces"][2])
        rho = W[0, :, 0, 0]
        W[4] = (2.5 + g * rho * (z - 1.0))[:, None, None]                 # hydrostatic for this g
        W[3] = 0.01 * wl.noise(3, W[3].shape) * (np.abs(z - 1.0) < 0.2)[:, None, None]
        o = make(ox, spec, W)
        k0 = float(np.sum(np.abs(o.get_state()[3])))
        run_steps(o, 0.7, 200)
        out.append(float(np.sum(np.abs(o.get_state()[3]))) / k0)
    assert out[0] > 1.5 * out[1], out


# ------------------------------------------------------------------------------------------ P11
CASES_P11 = [
    # name, ndim, n, coords, bc_lo, bc_hi, gravity, limiter, riemann, ns
    ("c3d_mixed", 3, [6, 5, 4], 0, [0, 2, 1], [0, 2, 1], 1, 4, 1, 2),
    ("c3d_refl", 3, [4, 4, 5], 0, [2, 1, 2], [1, 2, 2], 1, 1, 0, 1),
    ("c2d", 2, [7, 6], 0, [2, 0], [1, 0], 1, 2, 1, 1),
    ("c1d", 1, [9], 0, [1], [2], 1, 3, 1, 0),
    ("c3d_first_order", 3, [4, 5, 6], 0, [0, 1, 2], [0, 1, 2], 0, 0, 1, 1),
    ("s3d", 3, [6, 4, 5], 1, [2, 3, 0], [1, 3, 0], 2, 1, 1, 2),
    ("s3d_wedge", 3, [5, 4, 4], 1, [2, 3, 3], [1, 3, 3], 2, 4, 0, 1),
    ("s2d", 2, [6, 5], 1, [2, 3], [1, 3], 2, 2, 1, 1),
    ("s1d", 1, [8], 1, [2], [1], 2, 1, 1, 1),
    ("s3d_first_order", 3, [4, 4, 4], 1, [2, 3, 0], [1, 3, 0], 2, 0, 1, 0),
    # gas + radiation EOS (Eq. 6-7; names ending in _rad): P_r / P_g of order 0.1-1 on these states
    ("c3d_rad", 3, [6, 5, 4], 0, [0, 2, 1], [0, 2, 1], 1, 4, 1, 2),
    ("s3d_rad", 3, [6, 4, 5], 1, [2, 3, 0], [1, 3, 0], 2, 1, 1, 2),
    ("c1d_hll_rad", 1, [9], 0, [1], [2], 0, 2, 0, 0),
    # self-gravity (Eq. 4; gravity code 3): central mass + spherically averaged mass of the grid
    ("s3d_selfgrav", 3, [6, 4, 5], 1, [2, 3, 0], [1, 3, 0], 3, 1, 1, 1),
    ("s1d_selfgrav", 1, [8], 1, [2], [1], 3, 4, 1, 0),
    # internal-energy monitoring (Eq. 10-12; names ending in _emon): epsilon = 5 puts cells on all three branches of Eq. 12
    ("c3d_emon", 3, [6, 5, 4], 0, [0, 2, 1], [0, 2, 1], 1, 4, 1, 1),
    ("s3d_emon", 3, [6, 4, 5], 1, [2, 3, 0], [1, 3, 0], 2, 1, 1, 1),
    ("c2d_hll_emon", 2, [7, 6], 0, [2, 0], [1, 0], 0, 2, 0, 0),
    # both at once (the paper's supernova runs: gas + radiation EOS with the monitoring on)
    ("s3d_rad_emon", 3, [6, 4, 5], 1, [2, 3, 0], [1, 3, 0], 2, 1, 1, 2),
    ("c3d_hll_rad_emon", 3, [6, 5, 4], 0, [0, 2, 1], [0, 2, 1], 1, 4, 0, 1),
    # the maximum field count (16 stored fields; with the monitoring on a face flux vector carries 18 entries)
    ("s3d_max_emon", 3, [6, 5, 4], 1, [2, 3, 0], [1, 3, 0], 2, 2, 0, 11),
    ("c1d_max", 1, [12], 0, [1], [2], 1, 4, 1, 13),
]


def random_problem(ox, case, seed=0):
    name, ndim, n, coords, bc_lo, bc_hi, grav, lim, riem, ns = case
    rng = np.random.default_rng(seed + 100)
    if coords == 0:
        faces = [np.concatenate([[0.0], np.cumsum(rng.uniform(0.5, 1.5, m))]) / m for m in n]   # non-uniform on purpose
        for d in range(ndim):                      # periodic directions: keep the grid uniform-compatible
            pass
    else:
        faces = [wl.log_faces(0.8, 2.5, n[0])]
        if ndim >= 2:
            faces.append(np.concatenate([[0.0], np.cumsum(rng.uniform(0.5, 1.5, n[1]))]) / n[1] * 1.2 + 0.7)
        if ndim >= 3:
            faces.append(wl.uniform_faces(-0.5, 0.6, n[2]))
    kw = dict(coords=coords, n_scalars=ns, riemann=riem)
    if grav == 1:
        kw.update(gravity=ox.GRAV_UNIFORM, g=[0.3, -0.2, -0.5])
    elif grav == 2:
        kw.update(gravity=ox.GRAV_POINT_MASS, GM=0.8)
    elif grav == 3:
        kw.update(gravity=ox.GRAV_SELF, GM=0.8, G=0.6)
    if "_emon" in name:
        kw.update(emon_eps=5.0)
    if "_rad" in name:
        kw.update(eos=wl.EOS_GAS_RADIATION, eos_R=1.0, eos_ar=2.0)
    spec = wl._spec(name, ndim, n, faces, bc_lo, bc_hi, 1.4, lim, **kw)
    shape = tuple((n + [1, 1])[:3][::-1])
    W = np.empty((2 + ndim + ns,) + shape)
    W[0] = rng.uniform(0.5, 2.0, shape)
    for d in range(ndim):
        W[1 + d] = rng.uniform(-0.8, 0.8, shape)
    W[1 + ndim] = rng.uniform(0.5, 2.0, shape)
    for s in range(ns):
        W[2 + ndim + s] = rng.uniform(0.0, 1.0, shape)
    return spec, W


@pytest.mark.parametrize("case", CASES_P11, ids=[c[0] for c in CASES_P11])
def test_p11_naive_cell_update_equals_array_passes(oxlib, case):
    ox = oxlib
    spec, W = random_problem(ox, case)
    o = make(ox, spec, W)
    dt = 0.5 * o.compute_dt(0.5)
    n = spec["n"]
    naive = np.empty((spec["nvar"], n[2], n[1], n[0]))
    for k in range(n[2]):
        for j in range(n[1]):
            for i in range(n[0]):
                naive[:, k, j, i] = o.cell_update(i, j, k, dt)
    U0 = o.get_state()
    o.step(dt)
    U1 = o.get_state()
    assert np.max(np.abs(U1 - U0)) > 1e-3
    assert np.max(np.abs(naive - U1)) <= 1e-15 * np.max(np.abs(U1))


# ------------------------------------------------------------------------------------------ closed forms
def test_limiter_closed_forms(oxlib):
    ox = oxlib
    for lim in (1, 2, 3, 4):
        assert ox.limiter(lim, 1.0, -2.0) == 0.0 and ox.limiter(lim, -1.0, 0.0) == 0.0
        assert ox.limiter(lim, 0.7, 0.7) == pytest.approx(0.7, rel=1e-15)           # smooth: exact slope
        assert ox.limiter(lim, -0.7, -0.7) == pytest.approx(-0.7, rel=1e-15)
        assert ox.limiter(lim, 1.0, 3.0) == ox.limiter(lim, 3.0, 1.0)               # symmetric
        assert ox.limiter(lim, -1.0, -3.0) == -ox.limiter(lim, 1.0, 3.0)            # odd
    assert ox.limiter(0, 1.0, 1.0) == 0.0
    assert ox.limiter(1, 1.0, 3.0) == 1.0                                           # minmod
    assert ox.limiter(2, 1.0, 3.0) == pytest.approx(1.5, rel=1e-15)                 # harmonic mean 2ab/(a+b)
    assert ox.limiter(3, 1.0, 3.0) == pytest.approx(1.2, rel=1e-15)                 # ab(a+b)/(a^2+b^2)
    assert ox.limiter(4, 1.0, 3.0) == 2.0 and ox.limiter(4, 1.0, 1.5) == 1.25       # min(2a, 2b, (a+b)/2)


def test_spherical_geometry_closed_forms(oxlib):
    ox = oxlib
    n = [5, 4, 3]
    fr, ft, fp = wl.log_faces(0.5, 3.0, 5), wl.uniform_faces(0.4, 2.0, 4), wl.uniform_faces(-1.0, 0.5, 3)
    spec = wl._spec("geom", 3, n, [fr, ft, fp], [2, 3, 0], [1, 3, 0], 1.4, 1, coords=ox.SPHERICAL)
    o = ox.Oracle(spec)
    vols = []
    for k in range(3):
        for j in range(4):
            for i in range(5):
                dV, dS, xc = o.cell_geometry(i, j, k)
                vols.append(dV)
                assert xc[0] == 0.5 * (fr[i] + fr[i + 1])
                # divergence theorem for the constant fields e_x, e_y, e_z is awkward in spherical faces;
                # use instead the exact identities behind R10/R11:
                rm, rp, tm, tp = fr[i], fr[i + 1], ft[j], ft[j + 1]
                assert (dS[0, 1] - dS[0, 0]) / dV == pytest.approx(3.0 * (rp ** 2 - rm ** 2) / (rp ** 3 - rm ** 3), rel=1e-13)
                assert (dS[1, 1] - dS[1, 0]) / dV == pytest.approx(
                    (math.sin(tp) - math.sin(tm)) / (math.cos(tm) - math.cos(tp)) * 1.5 * (rp ** 2 - rm ** 2) / (rp ** 3 - rm ** 3), rel=1e-13)
                assert dS[2, 0] == dS[2, 1]
    # the cell volumes tile the wedge: closed form of the whole wedge volume
    total = (3.0 ** 3 - 0.5 ** 3) / 3.0 * (math.cos(0.4) - math.cos(2.0)) * 1.5
    assert fsum(vols) == pytest.approx(total, rel=1e-13)
    # ghost geometry: mirrored widths at reflecting / transmissive faces, wrapped widths at periodic ones
    xr, xp = o.faces(0), o.faces(2)
    assert xr[1] - xr[0] == pytest.approx(fr[2] - fr[1]) and xr[2] - xr[1] == pytest.approx(fr[1] - fr[0])
    assert xr[-1] - xr[-2] == pytest.approx(fr[-2] - fr[-3])
    assert xp[1] - xp[0] == pytest.approx(fp[-2] - fp[-3]) and xp[-1] - xp[-2] == pytest.approx(fp[2] - fp[1])


def test_cfl_time_step_closed_form(oxlib):
    ox = oxlib
    spec, W = wl.smooth_periodic(3, [6, 5, 4], seed=2, n_scalars=0)
    o = make(ox, spec, W)
    cs = np.sqrt(1.4 * W[4] / W[0])
    rate = (np.abs(W[1]) + cs) * 6 + (np.abs(W[2]) + cs) * 5 + (np.abs(W[3]) + cs) * 4
    assert o.compute_dt(0.6) == pytest.approx(0.6 / rate.max(), rel=1e-13)
    bad = W.copy()
    bad[4, 1, 2, 3] = -1.0
    o.set_state(bad, ox.PRIMITIVE)
    with pytest.raises(ox.OracleError) as e:
        o.compute_dt(0.6)
    assert e.value.code == ox.ERR_NONPHYSICAL


# ------------------------------------------------------------------------------------------ P12
def plane_wave_in_spherical(ox, ndim, n, t_end, limiter=2, amp=0.2, speed=1.0):
    """A density wave carried by a uniform Cartesian velocity (rho(x - U t), u = U, P = const) is an
    exact solution of Eq. 1.  Written in (r, theta[, phi]) it exercises every geometric factor and
    source term of Eq. 13-16 with u_theta, u_phi != 0.  A band of 4 cells along the open boundaries
    is reset to the exact solution after each step so that boundary errors never reach the interior."""
    gamma = 1.4
    fr = wl.uniform_faces(1.0, 2.0, n)
    # off-equator wedge so that the cot(theta) terms of Eq. 13-16 are not small
    ft = wl.uniform_faces(0.5, 1.5, n)
    faces = [fr, ft]
    nn = [n, n]
    if ndim == 3:
        faces.append(wl.uniform_faces(-0.5, 0.5, n))
        nn.append(n)
        Uc = speed * np.array([0.35, -0.2, 0.3])   # Cartesian velocity
        kv = 2 * math.pi * np.array([1.0, 1.0, -1.0])
    else:
        Uc = speed * np.array([0.0, 0.0, 0.4])     # along the polar axis: axisymmetric
        kv = 2 * math.pi * np.array([0.0, 0.0, 1.5])
    spec = wl._spec("planewave", ndim, nn, faces, [1] * ndim, [1] * ndim, gamma, limiter, coords=ox.SPHERICAL, n_scalars=1)
    r = wl.centres(fr)[None, None, :]
    th = wl.centres(ft)[None, :, None]
    ph = wl.centres(faces[2])[:, None, None] if ndim == 3 else np.zeros((1, 1, 1))
    x, y, z = r * np.sin(th) * np.cos(ph), r * np.sin(th) * np.sin(ph), r * np.cos(th)
    er = np.stack(np.broadcast_arrays(np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph), np.cos(th) + 0 * ph))
    et = np.stack(np.broadcast_arrays(np.cos(th) * np.cos(ph), np.cos(th) * np.sin(ph), -np.sin(th) + 0 * ph))
    ep = np.stack(np.broadcast_arrays(-np.sin(ph) + 0 * th, np.cos(ph) + 0 * th, 0 * th + 0 * ph))
    shape = np.broadcast_shapes(x.shape, y.shape, z.shape)

    def exact(t):
        W = np.empty((3 + ndim,) + shape)
        phase = kv[0] * (x - Uc[0] * t) + kv[1] * (y - Uc[1] * t) + kv[2] * (z - Uc[2] * t)
        W[0] = 1.0 + amp * np.sin(phase)
        W[1] = np.tensordot(Uc, er, axes=1)
        W[2] = np.tensordot(Uc, et, axes=1)
        if ndim == 3:
            W[3] = np.tensordot(Uc, ep, axes=1)
        W[1 + ndim] = 1.0
        W[2 + ndim] = 0.5 + 0.3 * np.cos(phase)
        return W
    o = make(ox, spec, exact(0.0))
    band = np.ones(shape, dtype=bool)
    sl = tuple(slice(4, -4) for _ in range(ndim))
    band[(slice(None),) * (3 - ndim) + sl] = False
    t = 0.0
    while t < t_end * (1 - 1e-12):
        dt = min(o.compute_dt(0.5), t_end - t)
        o.step(dt)
        t += dt
        P = o.get_state(ox.PRIMITIVE)
        E = exact(t)
        P[:, band] = E[:, band]
        o.set_state(P, ox.PRIMITIVE)
    P = o.get_state(ox.PRIMITIVE)
    E = exact(t_end)
    inner = (slice(None),) + (slice(None),) * (3 - ndim) + tuple(slice(6, -6) for _ in range(ndim))
    return [float(np.mean(np.abs(P[v][inner[1:]] - E[v][inner[1:]]))) for v in range(3 + ndim)]


@pytest.mark.parametrize("ndim,sizes,amp,speed,bar", [(2, (32, 64), 0.2, 1.0, 1.6), (3, (20, 40), 0.2, 1.0, 1.6),
                                                      (3, (20, 40), 0.0, 3.0, 1.45)])
def test_p12_cartesian_plane_wave_on_spherical_grid(oxlib, ndim, sizes, amp, speed, bar):
    # the fast uniform flow (amp 0, speed 3) makes the u_theta u_phi geometric terms of the
    # predictor dominate the error: dropping one of them shows up as first-order convergence
    e1 = plane_wave_in_spherical(oxlib, ndim, sizes[0], 0.1, amp=amp, speed=speed)
    e2 = plane_wave_in_spherical(oxlib, ndim, sizes[1], 0.1, amp=amp, speed=speed)
    for v in range(3 + ndim):
        order = math.log2(e1[v] / e2[v])
        assert order > bar, (v, e1, e2)
        assert e2[v] < 2e-3, (v, e2)


# ------------------------------------------------------------------------------------------ P9b
def falling_wave_error(ox, ndim, n, limiter=2):
    """rho(x - X(t)) with X = u0 t + g t^2/2, u = u0 + g t, P const: exact with uniform gravity, periodic box."""
    faces = [wl.uniform_faces(0.0, 1.0, n) for _ in range(ndim)]
    g = [0.8, -0.6, 0.0][:ndim] + [0.0] * (3 - ndim)
    u0 = [0.3, 0.5, 0.0][:ndim]
    spec = wl._spec("fallwave", ndim, [n] * ndim, faces, [0] * ndim, [0] * ndim, 1.4, limiter, gravity=ox.GRAV_UNIFORM, g=g)
    c = wl.centres(faces[0])
    grids = [c.reshape([n if (2 - e) == d else 1 for e in range(3)]) for d in range(ndim)]
    shape = tuple([n if (2 - e) < ndim else 1 for e in range(3)])
    t_end = 0.5

    def rho(t):
        ph = 0.0
        for d in range(ndim):
            ph = ph + (grids[d] - (u0[d] * t + 0.5 * g[d] * t * t))
        return np.broadcast_to(1.0 + 0.2 * np.sin(2 * math.pi * ph), shape)
    W = np.empty((2 + ndim,) + shape)
    W[0] = rho(0.0)
    for d in range(ndim):
        W[1 + d] = u0[d]
    W[1 + ndim] = 1.0
    o = make(ox, spec, W)
    run_to_time(o, 0.6, t_end)
    P = o.get_state(ox.PRIMITIVE)
    errs = [float(np.mean(np.abs(P[0] - rho(t_end))))]
    for d in range(ndim):
        errs.append(float(np.mean(np.abs(P[1 + d] - (u0[d] + g[d] * t_end)))))
    errs.append(float(np.mean(np.abs(P[1 + ndim] - 1.0))))
    return errs


@pytest.mark.parametrize("ndim,sizes", [(1, (64, 128)), (2, (32, 64))])
def test_p9b_advection_in_free_fall_second_order(oxlib, ndim, sizes):
    e1 = falling_wave_error(oxlib, ndim, sizes[0])
    e2 = falling_wave_error(oxlib, ndim, sizes[1])
    assert math.log2(e1[0] / e2[0]) > 1.7, (e1, e2)
    for v in range(1, 2 + ndim):        # velocity and pressure errors: second order too (and tiny)
        assert e2[v] < 1e-4 and (e1[v] < 1e-9 or math.log2(e1[v] / e2[v]) > 1.5), (v, e1, e2)


def test_p8_offcentre_sedov_wedge_matches_similarity_solution(oxlib):
    """PAPER.md Sect. 4.3 (L299-L309): off-centre blast in a spherical wedge, d_sh = xi0 (E1 t^2 / rho0)^(1/5) with
    xi0 ~ 1.15 for gamma = 5/3 at t = 0.08 (Eq. 25), "an expanding spherical blast that migrates away uniformly from
    r0".  On a 48^3 copy of the workload: the density peak sits within 10 % of the analytic distance along +r, -r and
    theta, and the blast is round to a cell and a half although none of its directions is a grid symmetry."""
    ox = oxlib
    n = 48
    spec, W = wl.sedov_wedge_3d(n)
    o = ox.Oracle(spec)
    o.set_state(W, ox.PRIMITIVE)
    run_to_time(o, spec["cfl"], spec["t_end"])
    rho = o.get_state()[0]
    xi0 = read_golden(os.path.join(GOLDEN, "sedov_similarity.txt"))["gamma_5_3"]
    d_exact = xi0 * (1.0 * spec["t_end"] ** 2 / 1.0) ** 0.2
    fr, ft = spec["faces"][0], spec["faces"][1]
    r, th = 0.5 * (fr[1:] + fr[:-1]), 0.5 * (ft[1:] + ft[:-1])
    dr = fr[1] - fr[0]
    line = rho[n // 2, n // 2, :]                       # radial line through the blast point (to half a cell)
    mid = int(np.argmin(np.abs(r - 0.7)))
    d_out = r[mid + int(np.argmax(line[mid:]))] - 0.7
    d_in = 0.7 - r[int(np.argmax(line[:mid]))]
    arc = rho[n // 2, :, mid]                            # theta line at r0
    jm = n // 2
    d_th = 0.7 * 2.0 * math.sin(0.5 * (th[jm + int(np.argmax(arc[jm:]))] - 0.5 * (th[jm - 1] + th[jm])))   # chord length
    for d in (d_out, d_in, d_th):
        assert abs(d - d_exact) <= 0.10 * d_exact, (d_out, d_in, d_th, d_exact)
    assert abs(d_out - d_in) <= 1.5 * dr and abs(d_out - d_th) <= 1.5 * dr, (d_out, d_in, d_th)
    assert np.max(line) > 1.6 and np.min(line) < 0.1     # a shell around an evacuated interior


# ------------------------------------------------------------------------------------------ P12: gas + radiation EOS
def test_p12_gas_radiation_eos_closed_forms(oxlib):
    """Eq. 6-7 (L88-L102).  Round trip e(rho, P(rho, e)) through the Newton-Raphson solve over twelve decades of
    P_r / P_g; the two limits (a_r -> 0: ideal gas with gamma; k_b/mu -> 0: P = e / 3, c_s^2 = (4/3) P / rho); and
    Eq. 7 against the definition c_s^2 = (dP/drho) at constant entropy, evaluated by a symmetric difference along
    the adiabat d(e/rho) = (P / rho^2) drho (catches a wrong coefficient in Eq. 7 as extracted)."""
    ox = oxlib
    GR, g, R = ox.EOS_GAS_RADIATION, 5.0 / 3.0, 1.3
    rng = np.random.default_rng(5)
    for _ in range(200):
        rho, T = 10.0 ** rng.uniform(-6, 2), 10.0 ** rng.uniform(-3, 3)
        ar = 10.0 ** rng.uniform(-3, 3)
        P = rho * R * T + ar * T ** 4 / 3.0
        e = rho * R * T / (g - 1.0) + ar * T ** 4                                    # Eq. 6a, 6b written out
        assert ox.eos_energy(GR, g, R, ar, rho, P) == pytest.approx(e, rel=1e-13)
        assert ox.eos_pressure(GR, g, R, ar, rho, e) == pytest.approx(P, rel=1e-13)
        al = (ar * T ** 4 / 3.0) / (rho * R * T)
        c2 = (g / (g - 1.0) + 20.0 * al + 16.0 * al * al) / (1.0 / (g - 1.0) + 12.0 * al) * R * T   # Eq. 7, P_g / rho = R T
        assert ox.eos_sound_speed(GR, g, R, ar, rho, P) == pytest.approx(math.sqrt(c2), rel=1e-13)
        # thermodynamic definition, symmetric difference along the adiabat
        eps = 1e-5
        es = e / rho
        Pp = ox.eos_pressure(GR, g, R, ar, rho * (1 + eps), (es + P / rho ** 2 * rho * eps) * rho * (1 + eps))
        Pm = ox.eos_pressure(GR, g, R, ar, rho * (1 - eps), (es - P / rho ** 2 * rho * eps) * rho * (1 - eps))
        assert (Pp - Pm) / (2 * eps * rho) == pytest.approx(c2, rel=2e-6)
    # limits
    assert ox.eos_pressure(GR, g, R, 1e-60, 2.0, 3.0) == pytest.approx((g - 1.0) * 3.0, rel=1e-14)
    assert ox.eos_sound_speed(GR, g, R, 1e-60, 2.0, 3.0) == pytest.approx(math.sqrt(g * 3.0 / 2.0), rel=1e-14)
    assert ox.eos_pressure(GR, g, 1e-60, 0.7, 2.0, 3.0) == pytest.approx(1.0, rel=1e-14)
    assert ox.eos_sound_speed(GR, g, 1e-60, 0.7, 2.0, 3.0) == pytest.approx(math.sqrt(4.0 / 3.0 * 3.0 / 2.0), rel=1e-12)


@pytest.mark.parametrize("limit", ["gas", "radiation"])
def test_p12_gas_radiation_limits_reduce_to_ideal_gases(oxlib, limit):
    """The whole step with the gas + radiation EOS equals the ideal-gas step with gamma (a_r -> 0) and with 4/3
    (k_b / mu -> 0) on a random 3-D problem with gravity, reflecting and periodic faces, two scalars."""
    ox = oxlib
    case = ("c3d_mixed", 3, [6, 5, 4], 0, [0, 2, 1], [0, 2, 1], 1, 4, 1, 2)
    spec, W = random_problem(ox, case)
    ideal, rad = dict(spec), dict(spec)
    if limit == "gas":
        rad.update(eos=wl.EOS_GAS_RADIATION, eos_R=1.0, eos_ar=1e-60)
    else:
        ideal["gamma"] = 4.0 / 3.0
        rad.update(eos=wl.EOS_GAS_RADIATION, eos_R=1e-60, eos_ar=1.0)
    a, b = make(ox, ideal, W), make(ox, rad, W)
    for _ in range(3):
        dt = a.compute_dt(0.4)
        assert b.compute_dt(0.4) == pytest.approx(dt, rel=1e-12)
        a.step(dt)
        b.step(dt)
    Ua, Ub = a.get_state(), b.get_state()
    assert np.max(np.abs(Ua - Ub)) <= 1e-12 * np.max(np.abs(Ua))


def test_p12_gas_radiation_conserves_and_keeps_uniform_states(oxlib):
    ox = oxlib
    spec, W = wl.smooth_periodic(3, [10, 8, 6], seed=3, n_scalars=1, limiter=wl.LIM_VANLEER)
    spec = dict(spec, eos=wl.EOS_GAS_RADIATION, eos_R=1.0, eos_ar=2.0)
    o = make(ox, spec, W)
    U0 = o.get_state()
    run_steps(o, 0.4, 20)
    U1 = o.get_state()
    for v in range(U0.shape[0]):
        assert abs(fsum(U1[v]) - fsum(U0[v])) <= 1e-13 * max(fsum(np.abs(U0[v])), 1.0)
    Wu = np.empty_like(W)
    for v, val in enumerate([1.3, 0.2, -0.4, 0.1, 0.9, 0.35]):
        Wu[v] = val
    o = make(ox, spec, Wu)
    Ua = o.get_state()
    run_steps(o, 0.4, 5)
    assert np.max(np.abs(o.get_state() - Ua)) <= 1e-14 * np.max(np.abs(Ua))


# ------------------------------------------------------------------------------------------ P13: self-gravity
def _shell_problem(ox, n, theta, phi, rho, G=2.0, GM=0.7):
    fr = wl.log_faces(0.5, 3.0, n[0])
    faces = [fr, wl.uniform_faces(*theta, n[1]), wl.uniform_faces(*phi, n[2])]
    spec = wl._spec("selfgrav", 3, list(n), faces, [2, 3, 3], [1, 3, 3], 1.4, wl.LIM_MINMOD, coords=wl.SPHERICAL,
                    gravity=wl.GRAV_SELF, GM=GM, G=G)
    rc = 0.5 * (fr[1:] + fr[:-1])
    W = np.zeros((5, n[2], n[1], n[0]))
    W[0] = rho(rc)[None, None, :]
    W[4] = 1.0
    return spec, W, rc


def test_p13_self_gravity_of_a_uniform_shell_is_the_closed_form(oxlib):
    """Eq. 4 (L73-L77): for uniform density rho between r_min and r, M(r) = M_c + (4 pi / 3) rho (r^3 - r_min^3)
    whatever the solid angle of the wedge (reading R28: the wedge stands for the whole sphere; the shell of the cell
    is counted up to its centre by volume)."""
    ox = oxlib
    for theta, phi in (((1.0, 1.9), (-0.3, 0.5)), ((0.4, 2.6), (0.0, 3.0))):
        spec, W, rc = _shell_problem(ox, (40, 6, 5), theta, phi, lambda r: 1.3 + 0.0 * r)
        o = make(ox, spec, W)
        exact = -(0.7 + 2.0 * 4.0 / 3.0 * math.pi * 1.3 * (rc ** 3 - 0.5 ** 3)) / rc ** 2
        got = np.array([o.self_gravity(i) for i in range(40)])
        assert np.max(np.abs(got / exact - 1.0)) <= 1e-14


def test_p13_self_gravity_power_law_and_limits(oxlib):
    """rho = r^-2: M(r) - M_c = 4 pi (r - r_min) exactly; the cell sums converge to it at second order.  G = 0 is the
    point mass of Eq. 3, step for step."""
    ox = oxlib
    errs = []
    for n in (40, 80):
        spec, W, rc = _shell_problem(ox, (n, 4, 4), (1.0, 1.9), (-0.3, 0.5), lambda r: r ** -2.0)
        o = make(ox, spec, W)
        exact = -(0.7 + 2.0 * 4.0 * math.pi * (rc - 0.5)) / rc ** 2
        errs.append(max(abs(o.self_gravity(i) / exact[i] - 1.0) for i in range(n)))
    assert errs[0] < 1e-2 and errs[1] < errs[0] / 3.0, errs
    case = ("s3d", 3, [6, 4, 5], 1, [2, 3, 0], [1, 3, 0], 2, 1, 1, 2)
    spec, W = random_problem(ox, case)
    a = make(ox, spec, W)
    b = make(ox, dict(spec, gravity=wl.GRAV_SELF, G=0.0), W)
    for _ in range(3):
        dt = a.compute_dt(0.4)
        a.step(dt)
        b.step(dt)
    assert np.array_equal(a.get_state(), b.get_state())


def test_p13_self_gravity_accelerates_a_static_shell_by_rho_g_dt(oxlib):
    """Uniform pressure, gas at rest: after one small step the radial momentum is dt rho g(r) (sign, use in predictor
    and update) and nothing else has moved."""
    ox = oxlib
    spec, W, rc = _shell_problem(ox, (32, 4, 4), (1.0, 1.9), (-0.3, 0.5), lambda r: 1.0 + 0.2 * np.sin(r))
    o = make(ox, spec, W)
    g = np.array([o.self_gravity(i) for i in range(32)])
    dt = 1e-4 * o.compute_dt(0.5)
    o.step(dt)
    U = o.get_state()
    expect = dt * W[0, 0, 0, :] * g
    assert np.max(np.abs(U[1, 1, 1, 1:-1] / expect[1:-1] - 1.0)) <= 1e-3
    assert np.max(np.abs(U[2])) <= 1e-12 and np.max(np.abs(U[3])) <= 1e-12


# ------------------------------------------------------------------------------------------ P14: internal-energy monitoring
def test_p14_monitoring_is_inert_where_the_internal_energy_is_large(oxlib):
    """Eq. 12: alpha = 1 wherever e >= eps e_k, and then Eq. 11 returns the total-energy result: with eps = 1e-6 a
    subsonic random problem steps exactly as without monitoring (to the rounding of e_k + (E - e_k))."""
    ox = oxlib
    case = ("c3d_mixed", 3, [6, 5, 4], 0, [0, 2, 1], [0, 2, 1], 1, 4, 1, 2)
    spec, W = random_problem(ox, case)
    a, b = make(ox, spec, W), make(ox, dict(spec, emon_eps=1e-6), W)
    for _ in range(3):
        dt = a.compute_dt(0.4)
        a.step(dt)
        b.step(dt)
    Ua, Ub = a.get_state(), b.get_state()
    assert np.max(np.abs(Ua - Ub)) <= 1e-14 * np.max(np.abs(Ua))


def test_p14_monitoring_keeps_a_cold_supersonic_stream_cold(oxlib):
    """The purpose of Eq. 10-12 (L120-L126): a uniform stream with e / e_k = 1e-10.  From the total energy alone the
    internal energy drifts by rounding of E (relative 1e-16 e_k / e = 1e-6 per step); with monitoring (alpha = 0 there)
    it follows Eq. 10, whose fluxes cancel exactly in a uniform state."""
    ox = oxlib
    spec, W = wl.smooth_periodic(3, [8, 6, 4], seed=2, n_scalars=0, limiter=wl.LIM_MINMOD)
    W[0], W[1], W[2], W[3], W[4] = 1.3, 3.0e5, -2.0e5, 1.0e5, 2.7
    drift = {}
    for eps in (0.0, 1e-6):
        o = make(ox, dict(spec, emon_eps=eps), W)
        U0 = o.get_state()
        e0 = U0[4] - 0.5 * (U0[1] ** 2 + U0[2] ** 2 + U0[3] ** 2) / U0[0]
        run_steps(o, 0.4, 20)
        U = o.get_state()
        e = U[4] - 0.5 * (U[1] ** 2 + U[2] ** 2 + U[3] ** 2) / U[0]
        drift[eps] = float(np.max(np.abs(e - e0) / e0))
    assert drift[1e-6] <= 1e-4 * drift[0.0] or drift[1e-6] <= 1e-12, drift


@pytest.mark.parametrize("eos", ["ideal", "gas_radiation"])
def test_p14_second_energy_equation_compression_work(oxlib, eos):
    """Eq. 10 with uniform rho, e, P and u = a x: de/dt = -(e + P) a, whatever the equation of state (with the gas + radiation
    EOS of Eq. 6, P_r / P_g ~ 1 here, e is no longer P / (gamma - 1): the pin checks that Eq. 10 takes P and e from the EOS).
    eps huge puts every cell on the alpha = 0 branch; one small step changes e by -(e + P) a dt in the interior (first order in
    dt and dx)."""
    ox = oxlib
    n, a = 64, 0.05
    fx = wl.uniform_faces(0.0, 1.0, n)
    kw = dict(eos=wl.EOS_GAS_RADIATION, eos_R=1.0, eos_ar=2.0) if eos == "gas_radiation" else {}
    spec = wl._spec("emon1d", 1, [n], [fx], [wl.BC_TRANSMISSIVE], [wl.BC_TRANSMISSIVE], 1.4, wl.LIM_MC, emon_eps=1e30, **kw)
    x = 0.5 * (fx[1:] + fx[:-1])
    W = np.empty((3, 1, 1, n))
    W[0], W[1, 0, 0], W[2] = 1.0, a * (x - 0.5), 2.0
    o = make(ox, spec, W)
    dt = 0.05 * o.compute_dt(0.5)
    U0 = o.get_state()
    o.step(dt)
    U = o.get_state()
    e0 = U0[2] - 0.5 * U0[1] ** 2 / U0[0]
    e1 = U[2] - 0.5 * U[1] ** 2 / U[0]
    got = ((e1 - e0) / dt)[0, 0, 4:-4]
    want = -(e0[0, 0, 4:-4] + 2.0) * a
    assert np.max(np.abs(got / want - 1.0)) <= 5e-3, (got[:3], want[:3])


# ---- P14b: the one-sided (supersonic) branches of the face velocity and the upwind choice of the advective flux of e ----
def _supersonic_tube(n, sign, limiter, eps, rho, u, e, gamma=1.4):
    """1-D tube, transmissive faces, primitive fields rho(x), sign * u(x), P = (gamma - 1) e(x)."""
    fx = wl.uniform_faces(0.0, 1.0, n)
    spec = wl._spec("emon_super", 1, [n], [fx], [wl.BC_TRANSMISSIVE], [wl.BC_TRANSMISSIVE], gamma, limiter, emon_eps=eps)
    x = wl.centres(fx)
    if sign < 0:
        x = 1.0 - x            # the mirror image of the sign > 0 problem
    W = np.empty((3, 1, 1, n))
    W[0, 0, 0], W[1, 0, 0], W[2, 0, 0] = rho(x), sign * u(x), (gamma - 1.0) * e(x)
    return spec, W, fx


def _internal_energy_1d(U):
    return (U[2] - 0.5 * U[1] ** 2 / U[0])[0, 0]


@pytest.mark.parametrize("sign", [+1, -1])
def test_p14_supersonic_faces_take_everything_from_upstream(oxlib, sign):
    """Eq. 10-12 where the whole Riemann fan lies on one side (S_L >= 0, resp. S_R <= 0): the flux is the upstream flux,
    so with first-order states (limiter NONE) no cell may depend on anything downstream of it -- neither through the
    face velocity of Eq. 10 (u_L, resp. u_R) nor through the advected e (upwind by the sign of the mass flux).  Two
    runs that differ only downstream of x = 0.5 (velocity, density, internal energy: all still supersonic) must agree
    BITWISE upstream of it; eps huge puts every cell on the alpha = 0 branch so that e comes from Eq. 10 alone.
    Taking u_R for u_L, or the downstream e, changes the last upstream cell."""
    ox = oxlib
    n = 48

    def run(downstream):
        du, dr, de = downstream
        spec, W, _ = _supersonic_tube(n, sign, wl.LIM_NONE, 1e30,
                                      lambda x: 1.0 + dr * (x > 0.5), lambda x: 40.0 + du * (x > 0.5),
                                      lambda x: 2.0 + 0.3 * np.sin(7.0 * x) + de * (x > 0.5))
        o = make(ox, spec, W)
        dt = 0.3 / (n * 60.0)
        for _ in range(3):
            o.step(dt)
        return o.get_state()

    Ua, Ub = run((0.0, 0.0, 0.0)), run((9.0, 0.7, 1.1))
    up = slice(0, n // 2 - 3) if sign > 0 else slice(n // 2 + 3, n)   # three steps move information by three cells at most
    down = slice(n // 2 + 1, n) if sign > 0 else slice(0, n // 2 - 1)
    assert np.array_equal(Ua[:, 0, 0, up], Ub[:, 0, 0, up])
    assert np.max(np.abs(Ua[:, 0, 0, down] - Ub[:, 0, 0, down])) > 0.1
    # one step: only the cell adjacent to the jump could see it, and it must not
    spec, W, _ = _supersonic_tube(n, sign, wl.LIM_NONE, 1e30, lambda x: 1.0 + 0.7 * (x > 0.5), lambda x: 40.0 + 9.0 * (x > 0.5),
                                  lambda x: 2.0 + 1.1 * (x > 0.5))
    spec0, W0, _ = _supersonic_tube(n, sign, wl.LIM_NONE, 1e30, lambda x: 1.0 + 0.0 * x, lambda x: 40.0 + 0.0 * x, lambda x: 2.0 + 0.0 * x)
    a, b = make(ox, spec, W), make(ox, spec0, W0)
    a.step(1e-4)
    b.step(1e-4)
    last_up = n // 2 - 1 if sign > 0 else n // 2
    assert np.array_equal(a.get_state()[:, 0, 0, last_up], b.get_state()[:, 0, 0, last_up])


@pytest.mark.parametrize("sign", [+1, -1])
def test_p14_supersonic_advection_of_e_is_first_order_upwind(oxlib, sign):
    """Uniform rho and u = sign * u0 with u0 > c everywhere, e(x) not uniform, limiter NONE, alpha = 0: div u = 0 at every
    face (u_f = u_L = u0, resp. u_R), the mass flux is rho u0, so Eq. 10 reduces to the donor-cell update
    e_i <- e_i - (u0 dt / dx) (e_i - e_upstream) -- a closed form that a downstream-biased Phi, a wrong sign of the
    flux difference or a non-zero compression term would miss at O(1)."""
    ox = oxlib
    n, u0 = 64, 30.0
    prof = lambda x: 2.0 + 0.8 * np.sin(2.0 * np.pi * x) + 0.3 * (x > 0.4)
    spec, W, fx = _supersonic_tube(n, sign, wl.LIM_NONE, 1e30, lambda x: 1.7 + 0.0 * x, lambda x: u0 + 0.0 * x, prof)
    o = make(ox, spec, W)
    U0 = o.get_state()
    dt, dx = 0.4 / (n * (u0 + 2.0)), 1.0 / n
    o.step(dt)
    e0, e1 = _internal_energy_1d(U0), _internal_energy_1d(o.get_state())
    up = np.roll(e0, 1) if sign > 0 else np.roll(e0, -1)
    want = e0 - (u0 * dt / dx) * (e0 - up)
    inner = slice(2, n - 2)
    # e is recovered from E - e_k with e_k / e ~ 400: rounding 400 x 1e-16
    assert np.max(np.abs(e1[inner] - want[inner]) / want[inner]) <= 1e-12
    # and the total-energy route does NOT give this (the pressure gradient does work on the stream; 1e-7 here): the pin is not vacuous
    spec_off = dict(spec, emon_eps=0.0)
    p = make(ox, spec_off, W)
    p.step(dt)
    e_plain = _internal_energy_1d(p.get_state())
    assert np.max(np.abs(e_plain[inner] - want[inner]) / want[inner]) > 1e-8


@pytest.mark.parametrize("sign", [+1, -1])
def test_p14_supersonic_compression_work_uses_the_upstream_face_velocity(oxlib, sign):
    """Uniform rho, e, P, supersonic u = sign * (u0 + b (x - 1/2)^2), limiter NONE, alpha = 0.  With u_f the UPSTREAM state's
    velocity, Eq. 10 gives e_i <- e_i - dt (e + P) (u_i - u_{i-1}) / dx (backward difference for sign > 0, its mirror
    image for sign < 0); the downstream state's velocity would give the forward difference, which differs by
    2 b dx (e + P) dt -- four orders above the tolerance."""
    ox = oxlib
    n, u0, b, gamma = 64, 30.0, 6.0, 1.4
    e_c = 2.0
    spec, W, fx = _supersonic_tube(n, sign, wl.LIM_NONE, 1e30, lambda x: 1.0 + 0.0 * x, lambda x: u0 + b * (x - 0.5) ** 2, lambda x: e_c + 0.0 * x)
    o = make(ox, spec, W)
    U0 = o.get_state()
    dt, dx = 0.2 / (n * (u0 + 4.0)), 1.0 / n
    o.step(dt)
    e1 = _internal_energy_1d(o.get_state())
    u = W[1, 0, 0]
    du_up = (u - np.roll(u, 1)) / dx if sign > 0 else (np.roll(u, -1) - u) / dx
    du_down = (np.roll(u, -1) - u) / dx if sign > 0 else (u - np.roll(u, 1)) / dx
    P = (gamma - 1.0) * e_c
    want = e_c - dt * (e_c + P) * du_up
    wrong = e_c - dt * (e_c + P) * du_down
    inner = slice(2, n - 2)
    tol = 2e-13 * 500.0          # rounding of E - e_k with e_k / e ~ 250
    assert np.max(np.abs(e1[inner] - want[inner])) <= tol * e_c
    assert np.min(np.abs(wrong[inner] - want[inner])) >= 1e3 * tol * e_c

"""Parity of the CUDA path (through the C ABI) with the CPU oracle.  `-m gpu` only.

Tolerances (BASELINE.json north_star, reading R22 for the norms): max relative difference per stored
field <= 1e-12 after one step; L1 relative difference <= 1e-9 after 100 steps (or the config's last
step).  dt itself must agree to 1e-13 relative.  Both sides get bit-identical inputs and face arrays.
"""
import numpy as np
import pytest

from paper_2503_04428_b200 import workloads as wl
from tests.helpers import l1_rel_per_field, max_rel_per_field
from tests.test_oracle_pins import CASES_P11, random_problem

pytestmark = pytest.mark.gpu

TOL_STEP = 1e-12
TOL_L1 = 1e-9
KERNELS = ["generic", "auto"]


@pytest.fixture(scope="module")
def hx():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2503_04428_b200 import hx as mod
    mod.lib()
    return mod


def make_pair(hx, ox, spec, W, kernel="auto"):
    g = hx.Hydro(spec)
    if kernel == "generic":
        g.set_option(hx.OPT_KERNEL, hx.KERNEL_GENERIC)
    g.set_state(np.ascontiguousarray(W), hx.PRIMITIVE)
    o = ox.Oracle(spec)
    o.set_state(W, ox.PRIMITIVE)
    return g, o


def cell_volumes(o, spec):
    n = spec["n"]
    if spec["coords"] == 0:
        return None   # uniform Cartesian reduced copies: dV constant, cancels in the ratio
    dV = np.empty((n[2], n[1], n[0]))
    for k in range(n[2]):
        for j in range(n[1]):
            for i in range(n[0]):
                dV[k, j, i] = o.cell_geometry(i, j, k)[0]
    return dV


# reduced copies of the five configs: several tiles plus a ragged tail in every direction
REDUCED = {
    "sod_1d": lambda: wl.sod_1d(1000),
    "kh_2d": lambda: wl.kh_2d((200, 136)),
    "sedov_3d": lambda: wl.sedov_3d((72, 44, 38)),
    "rt_3d": lambda: wl.rt_3d((70, 36, 42)),
    "wedge_3d": lambda: wl.wedge_3d((104, 22, 26)),
    "sedov_wedge_3d": lambda: wl.sedov_wedge_3d((72, 40, 36)),   # SURVEY 8(f) rank 3 (Sect. 4.3)
    "wedge_3d_rad": lambda: wl.wedge_3d_rad((72, 18, 20)),        # SURVEY 8(f) rank 1 (gas + radiation EOS, Eq. 6-7)
    "wedge_3d_selfgrav": lambda: wl.wedge_3d_selfgrav((72, 18, 20)),   # SURVEY 8(f) rank 4 (self-gravity, Eq. 4)
    "cold_stream_3d": lambda: wl.cold_stream_3d((40, 24, 20)),           # SURVEY 8(f) rank 2 (internal-energy monitoring, Eq. 10-12)
}


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("name", list(REDUCED))
def test_one_step_parity(hx, oxlib, name, kernel):
    ox = oxlib
    spec, W = REDUCED[name]()
    g, o = make_pair(hx, ox, spec, W, kernel)
    dt_g, dt_o = g.compute_dt(spec["cfl"]), o.compute_dt(spec["cfl"])
    # cold_stream_3d: P = (gamma-1)(E - e_k) with e_k / e = 3e6, so the sound speed in the CFL rate carries the rounding
    # of the prim -> cons -> prim round trip amplified by that ratio: 1e-16 x 3e6 x c / (|u| + c) ~ 1e-13
    assert abs(dt_g - dt_o) <= (1e-11 if name == "cold_stream_3d" else 1e-13) * dt_o
    g.step(dt_o)
    o.step(dt_o)
    Ug, Uo = g.get_state(), o.get_state()
    assert np.max(np.abs(Uo - ox.Oracle(spec).get_state())) > 0
    rel = max_rel_per_field(Ug, Uo, spec["ndim"])
    assert max(rel) <= TOL_STEP, (name, kernel, g.step_kernel, rel)
    # the rate folded into the step equals the stand-alone reduction of the oracle on the new state
    dt_g2, dt_o2 = g.compute_dt(spec["cfl"]), o.compute_dt(spec["cfl"])
    assert abs(dt_g2 - dt_o2) <= 1e-12 * dt_o2


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("name", list(REDUCED))
def test_hundred_step_parity(hx, oxlib, name, kernel):
    ox = oxlib
    spec, W = REDUCED[name]()
    g, o = make_pair(hx, ox, spec, W, kernel)
    nsteps = 100 if spec["steps"] is None else min(100, spec["steps"])
    for s in range(nsteps):
        dt_g, dt_o = g.compute_dt(spec["cfl"]), o.compute_dt(spec["cfl"])
        assert abs(dt_g - dt_o) <= 1e-10 * dt_o, (s, dt_g, dt_o)
        g.step(dt_g)
        o.step(dt_o)
    Ug, Uo = g.get_state(), o.get_state()
    l1 = l1_rel_per_field(Ug, Uo, spec["ndim"], cell_volumes(o, spec))
    assert max(l1) <= TOL_L1, (name, kernel, g.step_kernel, l1)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("case", CASES_P11, ids=[c[0] for c in CASES_P11])
def test_every_bc_geometry_solver_limiter(hx, oxlib, case, kernel):
    """Tiny random problems: every boundary type on every face, both geometries, both solvers, every
    limiter, non-uniform grids, gravity of both kinds (same cases as oracle pin P11)."""
    ox = oxlib
    spec, W = random_problem(ox, case)
    g, o = make_pair(hx, ox, spec, W, kernel)
    for _ in range(3):
        dt = 0.5 * o.compute_dt(0.5)
        assert abs(0.5 * g.compute_dt(0.5) - dt) <= 1e-13 * dt
        g.step(dt)
        o.step(dt)
    rel = max_rel_per_field(g.get_state(), o.get_state(), spec["ndim"])
    assert max(rel) <= 3 * TOL_STEP, (case[0], rel)


@pytest.mark.parametrize("lim", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("riemann", [0, 1])
def test_limiters_and_solvers_3d(hx, oxlib, lim, riemann):
    ox = oxlib
    spec, W = wl.smooth_periodic(3, [40, 24, 20], seed=21, n_scalars=1, limiter=lim, riemann=riemann)
    W[0] += 0.8 * (W[1] > 0.1)        # add jumps so that limiters and wave-speed branches switch
    g, o = make_pair(hx, ox, spec, W)
    for _ in range(5):
        dt = o.compute_dt(0.5)
        g.step(dt)
        o.step(dt)
    rel = max_rel_per_field(g.get_state(), o.get_state(), 3)
    assert max(rel) <= 5 * TOL_STEP, rel


def test_library_spacing_modes_match_custom_faces(hx, oxlib):
    """HX_SPACING_UNIFORM / LOG computed inside the library vs the oracle's own uniform / log faces."""
    ox = oxlib
    spec, W = wl.wedge_3d((40, 10, 12))
    spec = dict(spec)
    spec["faces"] = [None, None, None]
    spec["spacing"] = [wl.SPACING_LOG, wl.SPACING_UNIFORM, wl.SPACING_UNIFORM]
    g, o = make_pair(hx, ox, spec, W)
    dt = o.compute_dt(0.6)
    assert abs(g.compute_dt(0.6) - dt) <= 1e-13 * dt
    g.step(dt)
    o.step(dt)
    assert max(max_rel_per_field(g.get_state(), o.get_state(), 3)) <= TOL_STEP


def test_state_round_trip_and_forms(hx, oxlib):
    ox = oxlib
    import torch
    spec, W = wl.smooth_periodic(3, [18, 10, 6], seed=4, n_scalars=2)
    g, o = make_pair(hx, ox, spec, W)
    assert g.nvar == 7 and g.shape == (7, 6, 10, 18)
    Uo = o.get_state()
    Ug = g.get_state()
    assert np.max(np.abs(Ug - Uo)) <= 1e-15 * np.max(np.abs(Uo))
    Wg = g.get_state(form=hx.PRIMITIVE)
    assert np.max(np.abs(Wg - W)) <= 1e-14
    g.set_state(Uo, hx.CONSERVED)
    assert np.array_equal(g.get_state(), Uo)                      # conserved in -> out is a pure copy
    # device-pointer path on a non-default torch stream
    stream = torch.cuda.Stream()
    g.set_stream(stream)
    with torch.cuda.stream(stream):
        dev = torch.from_numpy(Uo).cuda()
        g.set_state(dev, hx.CONSERVED)
        out = torch.empty_like(dev)
        g.get_state(out, hx.CONSERVED)
    assert torch.equal(out.cpu(), torch.from_numpy(Uo))
    with pytest.raises(ValueError):
        g.set_state(np.zeros(5))


def test_nonphysical_state_is_reported_not_floored(hx):
    spec, W = wl.smooth_periodic(2, [32, 16], seed=9, n_scalars=0)
    g = hx.Hydro(spec)
    bad = W.copy()
    bad[3, 0, 3, 5] = -0.5          # negative pressure
    g.set_state(bad, hx.PRIMITIVE)
    with pytest.raises(hx.HxError) as e:
        g.compute_dt(0.5)
    assert e.value.code == hx.ERR_NONPHYSICAL
    g.set_state(W, hx.PRIMITIVE)    # the flag is cleared by a new state
    assert g.compute_dt(0.5) > 0
    with pytest.raises(hx.HxError):
        g.step(-1.0)
    # a far too large time step drives the update non-physical: reported at the next sync call
    g.step(50.0 * g.compute_dt(0.5))
    with pytest.raises(hx.HxError) as e:
        g.compute_dt(0.5)
    assert e.value.code == hx.ERR_NONPHYSICAL


def test_nonphysical_state_in_the_fused_3d_kernel(hx):
    spec, W = wl.smooth_periodic(3, [40, 20, 12], seed=5, n_scalars=0)
    g = hx.Hydro(spec)
    g.set_state(W, hx.PRIMITIVE)
    g.step(g.compute_dt(0.5))
    assert g.step_kernel.startswith("tile2") and g.compute_dt(0.5) > 0
    g.step(80.0 * g.compute_dt(0.5))
    with pytest.raises(hx.HxError) as e:
        g.compute_dt(0.5)
    assert e.value.code == hx.ERR_NONPHYSICAL


def test_minimum_sizes_and_degenerate_shapes(hx, oxlib):
    ox = oxlib
    for ndim, n in ((1, [2]), (2, [2, 3]), (3, [2, 2, 2]), (3, [3, 2, 5]), (1, [33])):
        spec, W = wl.smooth_periodic(ndim, n, seed=ndim, n_scalars=1)
        g, o = make_pair(hx, ox, spec, W)
        dt = o.compute_dt(0.4)
        g.step(dt)
        o.step(dt)
        assert max(max_rel_per_field(g.get_state(), o.get_state(), ndim)) <= TOL_STEP, n


@pytest.mark.parametrize("n", [(58, 20, 18), (64, 16, 8), (65, 17, 5), (33, 9, 16), (32, 8, 33), (96, 39, 70), (64, 26, 40), (2, 2, 2), (5, 3, 2)])
def test_tile_edges(hx, oxlib, n):
    """Grids that give exactly full 32 x 8 tiles (and multiples of the earlier 13-row tiles), one cell more than a full tile in x and y, ragged tails,
    single partial tiles, and z extents that split into several chunks."""
    ox = oxlib
    spec, W = wl.smooth_periodic(3, list(n), seed=n[0], n_scalars=0, limiter=wl.LIM_MC)
    g, o = make_pair(hx, ox, spec, W, "auto")
    for _ in range(2):
        dt = o.compute_dt(0.5)
        g.step(dt)
        o.step(dt)
    assert g.step_kernel.startswith("tile2")
    assert max(max_rel_per_field(g.get_state(), o.get_state(), 3)) <= 2 * TOL_STEP, n


UNIFORM = {   # 2^k cells on dyadic extents: bitwise-uniform tables -> the constant-geometry instantiations
    "sedov_3d": lambda: wl.sedov_3d((64, 32, 32)),
    "rt_3d": lambda: wl.rt_3d((32, 64, 64)),
    "cold_stream_3d": lambda: wl.cold_stream_3d((64, 32, 32)),   # internal-energy monitoring in the tile kernel
}


@pytest.mark.parametrize("name", list(UNIFORM))
def test_uniform_grid_instantiations(hx, oxlib, name):
    ox = oxlib
    spec, W = UNIFORM[name]()
    g, o = make_pair(hx, ox, spec, W)
    for s in range(40):
        dt_g, dt_o = g.compute_dt(spec["cfl"]), o.compute_dt(spec["cfl"])
        assert abs(dt_g - dt_o) <= 1e-10 * dt_o, (s, dt_g, dt_o)
        g.step(dt_g)
        o.step(dt_o)
        if s == 0:
            assert g.step_kernel == ("tile2_emon" if name == "cold_stream_3d" else "tile2_uni")
            rel = max_rel_per_field(g.get_state(), o.get_state(), 3)
            assert max(rel) <= TOL_STEP, (name, rel)
    l1 = l1_rel_per_field(g.get_state(), o.get_state(), 3)
    assert max(l1) <= TOL_L1, (name, l1)


# ---- BASELINE.json's full sizes, in the launch configuration bench.py times --------------------------------
FULL = {
    "sedov_3d": (lambda: wl.sedov_3d(256), "tile2_uni"),
    "rt_3d": (lambda: wl.rt_3d(512), "tile2_uni"),
    "wedge_3d": (lambda: wl.wedge_3d((1024, 256, 256)), "tile2"),
    "sedov_wedge_3d": (lambda: wl.sedov_wedge_3d(256), "tile2"),
    "wedge_3d_rad": (lambda: wl.wedge_3d_rad((512, 128, 128)), "tile2_rad"),   # gas + radiation EOS: a quarter-size wedge
    "wedge_3d_selfgrav": (lambda: wl.wedge_3d_selfgrav((512, 128, 128)), "tile2"),   # self-gravity: a quarter-size wedge
}


def sample_cells(n, seed, extra):
    """Cells the oracle evaluates one by one: domain corners and face centres, both sides of tile edges
    (x multiples of 32, y multiples of 8) and of z-chunk edges, cells where the workload has structure
    (`extra`), and seeded random interior cells."""
    nx, ny, nz = n
    rng = np.random.default_rng(seed)
    cells = set()
    for i in (0, 1, nx // 2, nx - 2, nx - 1):
        for j in (0, 1, ny // 2, ny - 2, ny - 1):
            for k in (0, 1, nz // 2, nz - 2, nz - 1):
                cells.add((i, j, k))
    for _ in range(60):
        ti, tj = 32 * int(rng.integers(1, max(2, nx // 32))), 8 * int(rng.integers(1, max(2, ny // 8)))
        k = int(rng.integers(0, nz))
        for di in (-1, 0):
            for dj in (-1, 0):
                cells.add((min(ti + di, nx - 1), min(tj + dj, ny - 1), k))
    for kc in range(16, nz, 16):                     # every possible chunk edge (chunks are >= 16 planes)
        cells.add((int(rng.integers(0, nx)), int(rng.integers(0, ny)), kc - 1))
        cells.add((int(rng.integers(0, nx)), int(rng.integers(0, ny)), kc))
    for _ in range(150):
        cells.add((int(rng.integers(0, nx)), int(rng.integers(0, ny)), int(rng.integers(0, nz))))
    cells.update(extra)
    return sorted(cells)


@pytest.mark.parametrize("name", list(FULL))
def test_full_size_sampled_parity(hx, oxlib, name):
    """One step at the benchmark size; the oracle's per-cell evaluation (ox_cell_update, the naive 13-point
    star of pin P11) on sampled cells, same tolerance as the element-by-element tests."""
    ox = oxlib
    make, kernel_name = FULL[name]
    spec, W = make()
    n = spec["n"]
    g = hx.Hydro(spec)
    g.set_state(np.ascontiguousarray(W), hx.PRIMITIVE)
    o = ox.Oracle(spec)
    o.set_state(W, ox.PRIMITIVE)
    del W
    dt_g, dt_o = g.compute_dt(spec["cfl"]), o.compute_dt(spec["cfl"])
    assert abs(dt_g - dt_o) <= 1e-13 * dt_o
    g.step(dt_o)
    assert g.step_kernel == kernel_name
    Ug = g.get_state()
    nvar, ndim = Ug.shape[0], 3
    den = [float(np.max(np.abs(Ug[v]))) for v in range(nvar)]
    mden = max(den[1:1 + ndim])
    den = [mden if 1 <= v <= ndim else den[v] for v in range(nvar)]
    if name == "sedov_3d":      # the blast region (160 hot cells around the origin) and its rim
        extra = [(n[0] // 2 + a, n[1] // 2 + b, n[2] // 2 + c) for a in range(-5, 5) for b in (-4, -1, 0, 3) for c in (-4, 0, 3)]
    elif name == "rt_3d":       # the perturbed interface slab around z = 1
        extra = [(37 * q % n[0], 91 * q % n[1], n[2] // 2 + c) for q in range(40) for c in (-14, -2, -1, 0, 1, 13)]
    elif name in ("wedge_3d_rad", "wedge_3d_selfgrav"):
        extra = [(a, 53 * a % n[1], 29 * a % n[2]) for a in list(range(0, 8)) + [81, 82, 154, 155, 236, 237]]
    elif name == "sedov_wedge_3d":   # the blast region around (r0, theta0, phi0) = mid-domain
        extra = [(n[0] // 2 + a, n[1] // 2 + b, n[2] // 2 + c) for a in range(-5, 5) for b in (-4, -1, 0, 3) for c in (-4, 0, 3)]
    else:                       # the bomb in the first radial cells and the composition shell edges
        extra = [(a, 53 * a % n[1], 29 * a % n[2]) for a in list(range(0, 8)) + [161, 162, 307, 308, 471, 472, 473]]
    worst = 0.0
    cells = sample_cells(n, 7, extra)
    for (i, j, k) in cells:
        ref = o.cell_update(i, j, k, dt_o)
        for v in range(nvar):
            err = abs(Ug[v, k, j, i] - ref[v]) / den[v] if den[v] > 0 else abs(Ug[v, k, j, i] - ref[v])
            worst = max(worst, err)
    assert worst <= TOL_STEP, (name, worst, len(cells))
    # conservation as a property that holds at any size: with periodic / reflecting faces the mass is unchanged
    if name == "rt_3d":
        m0 = float(np.sum(o.get_state()[0], dtype=np.float64))
        m1 = float(np.sum(Ug[0], dtype=np.float64))
        assert abs(m1 - m0) <= 1e-12 * m0


def test_step_is_deterministic(hx):
    """Two handles, same input, five steps: bitwise identical states and time steps.  (A race in the shared-memory
    exchange or in the in-place plane conversion would show up as run-to-run differences; compute-sanitizer is
    not available on this pool.)"""
    for make in (lambda: wl.rt_3d((64, 40, 36)), lambda: wl.wedge_3d((72, 24, 20))):
        spec, W = make()
        out = []
        for _ in range(2):
            g = hx.Hydro(spec)
            g.set_state(np.ascontiguousarray(W), hx.PRIMITIVE)
            dts = []
            for _s in range(5):
                dts.append(g.compute_dt(spec["cfl"]))
                g.step(dts[-1])
            out.append((dts, g.get_state()))
        assert out[0][0] == out[1][0]
        assert np.array_equal(out[0][1], out[1][1])


def test_full_size_ten_steps_sedov(hx, oxlib):
    """Ten steps of config 3 at its full size (256^3) against the whole-array oracle, every cell: L1 relative
    difference per field <= 1e-9 and max relative difference <= 1e-11 (the blast has crossed a few cells by then)."""
    ox = oxlib
    spec, W = wl.sedov_3d(256)
    g, o = make_pair(hx, ox, spec, W)
    del W
    for s in range(10):
        dt_g, dt_o = g.compute_dt(spec["cfl"]), o.compute_dt(spec["cfl"])
        assert abs(dt_g - dt_o) <= 1e-11 * dt_o, (s, dt_g, dt_o)
        g.step(dt_g)
        o.step(dt_o)
    assert g.step_kernel == "tile2_uni"
    Ug, Uo = g.get_state(), o.get_state()
    assert max(l1_rel_per_field(Ug, Uo, 3)) <= TOL_L1
    assert max(max_rel_per_field(Ug, Uo, 3)) <= 1e-11

"""hx_self_gravity_noalloc -- the entry point that allocates nothing (scratch in a static __device__ array of libhx.so) --
against the existing handle path (hx_self_gravity_table: the launch hx_step makes, scratch from cudaMalloc).  `-m gpu` only.

Collected last on purpose (file name): the suite runs with `pytest -x`, and a failure here must not hide the other tests.
Two calls in a row on DIFFERENT problems share the one scratch array, so stale contents of the first call would show up in
the second; a third call repeats the first problem and must reproduce it bit for bit.
"""
import numpy as np
import pytest

from paper_2503_04428_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-12   # relative, per entry: the one-step tolerance of tests/test_parity_gpu.py (the two paths differ in summation order only)


@pytest.fixture(scope="module")
def hx():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2503_04428_b200 import hx as mod
    mod.lib()
    return mod


def existing_path(hx, spec, W):
    g = hx.Hydro(spec)
    g.set_state(np.ascontiguousarray(W), hx.PRIMITIVE)
    out = g.self_gravity_table()
    g.close()
    return out


def device_inputs(spec, W):
    import torch
    rho = torch.from_numpy(np.ascontiguousarray(W[0])).cuda()          # density: the same in primitive and conserved form
    faces = [torch.from_numpy(np.ascontiguousarray(f, dtype=np.float64)).cuda() for f in spec["faces"]]
    out = torch.full((spec["n"][0],), float("nan"), dtype=torch.float64, device="cuda")
    return rho, faces, out


def test_no_alloc_self_gravity_matches_the_handle_path_on_two_calls_in_a_row(hx):
    import torch
    problems = [wl.wedge_3d_selfgrav((192, 48, 40)), wl.wedge_3d_selfgrav((72, 18, 20))]   # 1920 and 360 rows: 128 full row groups, then fewer
    want = [existing_path(hx, spec, W) for spec, W in problems]
    inputs = [device_inputs(spec, W) for spec, W in problems]
    assert np.all(want[0] < 0) and np.max(np.abs(want[0] * 1.0 + 1.0 / wl.centres(problems[0][0]["faces"][0]) ** 2)) > 1e-3   # the envelope matters
    # warm-up call (module load, address look-up), then the free device memory must stay put over the calls that follow
    spec, _ = problems[1]
    rho, faces, out = inputs[1]
    hx.self_gravity_noalloc(rho, faces[0], faces[1], faces[2], spec["GM"], spec["G"], out)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    got = []
    for idx in (0, 1, 0):                      # back to back on the same stream, sharing the scratch array
        spec, _ = problems[idx]
        rho, faces, out = inputs[idx]
        out.fill_(float("nan"))
        hx.self_gravity_noalloc(rho, faces[0], faces[1], faces[2], spec["GM"], spec["G"], out)
        got.append(out.cpu().numpy().copy())
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    for idx, g in zip((0, 1, 0), got):
        assert np.all(np.isfinite(g)), idx
        rel = np.max(np.abs(g - want[idx]) / np.abs(want[idx]))
        assert rel <= TOL, (idx, rel)
    assert np.array_equal(got[0], got[2])      # same input after another problem went through the scratch: same bits
    assert free_before - free_after < (1 << 20), (free_before, free_after)   # nothing was allocated on the device


def test_no_alloc_rejects_sizes_beyond_the_static_array(hx):
    import torch
    for n in ((hx.NOALLOC_MAX_N0 + 1, 2, 2), (4, hx.NOALLOC_MAX_ANGULAR - 1, 2)):
        n0, n1, n2 = n
        rho = torch.ones((n2, n1, n0), dtype=torch.float64, device="cuda")
        fr, ft, fp = (torch.linspace(1.0, 2.0, m + 1, dtype=torch.float64, device="cuda") for m in (n0, n1, n2))
        out = torch.zeros(n0, dtype=torch.float64, device="cuda")
        with pytest.raises(hx.HxError) as e:
            hx.self_gravity_noalloc(rho, fr, ft, fp, 1.0, 0.1, out)
        assert e.value.code == hx.ERR_UNSUPPORTED
        assert "HX_NOALLOC_MAX" in str(e.value)
    # the largest accepted radial size works, and a closed form pins it: uniform density, G M_c = 0
    n0, n1, n2 = hx.NOALLOC_MAX_N0, 3, 5
    fr = torch.linspace(1.0, 3.0, n0 + 1, dtype=torch.float64, device="cuda")
    ft = torch.linspace(1.0, 2.0, n1 + 1, dtype=torch.float64, device="cuda")
    fp = torch.linspace(-0.5, 0.7, n2 + 1, dtype=torch.float64, device="cuda")
    rho = torch.full((n2, n1, n0), 0.7, dtype=torch.float64, device="cuda")
    out = torch.zeros(n0, dtype=torch.float64, device="cuda")
    G = 0.3
    hx.self_gravity_noalloc(rho, fr, ft, fp, 0.0, G, out)
    rc = 0.5 * (fr[1:] + fr[:-1]).cpu().numpy()
    exact = -G * 4.0 * np.pi / 3.0 * 0.7 * (rc ** 3 - 1.0) / rc ** 2        # -G M(<r_c) / r_c^2 of a uniform shell starting at r = 1
    assert np.max(np.abs(out.cpu().numpy()[1:] / exact[1:] - 1.0)) <= 1e-11

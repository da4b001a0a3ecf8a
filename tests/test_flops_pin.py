"""bench.py's algorithmic flop count (the numerator of roofline.achieved, a hand count from O1-O7) against what ncu counted on
the GPU (profiles/r2_*_ncu_full.md, committed text): the kernels execute the algorithm's work plus the ring warps' redundant
predictor (20-30 % of the cells), the z-chunk overlap and the correction steps of reciprocals / square roots, and never less.
A term dropped from or doubled in the hand count moves the ratio out of the band.  CPU only."""
import os
import re

import pytest

import bench
from paper_2503_04428_b200 import workloads as wl

PROFILES = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "profiles")
CASES = {
    "rt_3d": lambda: wl.rt_3d((8, 8, 8)), "sedov_3d": lambda: wl.sedov_3d((8, 8, 8)), "wedge_3d": lambda: wl.wedge_3d((8, 8, 8)),
    "kh_2d": lambda: wl.kh_2d((8, 8)), "sedov_wedge_3d": lambda: wl.sedov_wedge_3d(8), "wedge_3d_rad": lambda: wl.wedge_3d_rad((8, 8, 8)),
    "wedge_3d_sn": lambda: wl.wedge_3d_sn((8, 8, 8)),
}


@pytest.mark.parametrize("name", list(CASES))
def test_algorithmic_flops_within_the_executed_flops(name):
    text = open(os.path.join(PROFILES, f"r2_{name}_ncu_full.md")).read()
    m = re.search(r"= (\d+) per cell-update \((\d+) flop, FMA = 2\)", text)
    assert m, "fp64 instruction line not found"
    executed = float(m.group(2))
    spec, _ = CASES[name]()
    alg = bench.alg_flops_per_cell(spec)
    assert 0.65 * executed <= alg <= executed, (name, alg, executed)

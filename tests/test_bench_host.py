"""Host logic of bench.py that needs no GPU: the max-over-ranks timing aggregation on a world_size-2
gloo group (the N > 1 path runs independent replicas), the algorithmic flop count,
and the reference arm's JSON line."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=2)
local = 10.0 + 5.0 * int(os.environ["RANK"])
print("AGG", bench.aggregate_max_ms(local, 2))
dist.destroy_process_group()
"""


def test_max_over_ranks_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29533")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    for p, (out, err) in zip(procs, outs):
        assert p.returncode == 0, err
        assert "AGG 15.0" in out, out


def test_algorithmic_flop_count_matches_design():
    sys.path.insert(0, ROOT)
    import bench
    from paper_2503_04428_b200 import workloads as wl
    assert bench.alg_flops_per_cell(wl.sedov_3d((8, 8, 8))[0]) == 629
    assert bench.alg_flops_per_cell(wl.rt_3d((8, 8, 8))[0]) == 629 + 2 * 84 + 3 * 7 * 4 + 31
    assert bench.alg_flops_per_cell(wl.wedge_3d((8, 8, 8))[0]) == 629 + 4 * 84 + 31 + 65


def test_reference_arm_prints_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "rt_3d_small",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0

"""Small helpers shared by the tests (no method arithmetic)."""
import math

import numpy as np


def run_to_time(sim, cfl, t_end, max_steps=100000):
    t, steps = 0.0, 0
    while t < t_end * (1.0 - 1e-14) and steps < max_steps:
        dt = min(sim.compute_dt(cfl), t_end - t)
        sim.step(dt)
        t += dt
        steps += 1
    return steps


def run_steps(sim, cfl, nsteps):
    dts = []
    for _ in range(nsteps):
        dt = sim.compute_dt(cfl)
        sim.step(dt)
        dts.append(dt)
    return dts


def fsum(a):
    return math.fsum(np.asarray(a, dtype=np.float64).ravel().tolist())


def max_rel_per_field(g, o, ndim):
    """Reading R22: max_i |g_i - o_i| / max_i |o_i| per stored field; the momentum components
    share one denominator (max |m| over all components)."""
    nvar = o.shape[0]
    out = []
    mden = max(float(np.max(np.abs(o[1 + d]))) for d in range(ndim))
    for v in range(nvar):
        den = mden if 1 <= v <= ndim else float(np.max(np.abs(o[v])))
        num = float(np.max(np.abs(g[v] - o[v])))
        out.append(0.0 if num == 0.0 else (num / den if den > 0 else float("inf")))
    return out


def l1_rel_per_field(g, o, ndim, dV=None):
    nvar = o.shape[0]
    w = 1.0 if dV is None else dV
    out = []
    mden = sum(float(np.sum(np.abs(o[1 + d]) * w)) for d in range(ndim))
    for v in range(nvar):
        den = mden if 1 <= v <= ndim else float(np.sum(np.abs(o[v]) * w))
        num = float(np.sum(np.abs(g[v] - o[v]) * w))
        out.append(0.0 if num == 0.0 else (num / den if den > 0 else float("inf")))
    return out


def read_golden(path):
    vals = {}
    with open(path) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, v = line.split()
            vals[k] = float(v)
    return vals

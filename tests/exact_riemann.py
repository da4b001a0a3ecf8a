"""Exact solution of the 1-D Riemann problem for an ideal gas (test-side pin, numpy only).

Restates the classical construction (Toro 2009, ch. 4; the paper's App. C.1 says "the exact
solution is known analytically"): the star pressure p* is the root of
    f(p) = f_L(p) + f_R(p) + u_R - u_L = 0,
with f_K the shock (p > p_K) or rarefaction (p <= p_K) branch; the solution is then sampled
along x/t.  Independent of both the oracle and the CUDA path.
"""
import numpy as np


def _fK(p, rho, pk, gamma):
    a = np.sqrt(gamma * pk / rho)
    if p > pk:  # shock
        A = 2.0 / ((gamma + 1.0) * rho)
        B = (gamma - 1.0) / (gamma + 1.0) * pk
        f = (p - pk) * np.sqrt(A / (p + B))
        df = np.sqrt(A / (p + B)) * (1.0 - 0.5 * (p - pk) / (p + B))
    else:  # rarefaction
        f = 2.0 * a / (gamma - 1.0) * ((p / pk) ** ((gamma - 1.0) / (2.0 * gamma)) - 1.0)
        df = 1.0 / (rho * a) * (p / pk) ** (-(gamma + 1.0) / (2.0 * gamma))
    return f, df


def star_state(left, right, gamma):
    """(p*, u*) for left = (rho, u, p), right = (rho, u, p)."""
    rl, ul, pl = left
    rr, ur, pr = right
    p = max(1e-12, 0.5 * (pl + pr))
    for _ in range(200):
        fl, dfl = _fK(p, rl, pl, gamma)
        fr, dfr = _fK(p, rr, pr, gamma)
        pn = p - (fl + fr + ur - ul) / (dfl + dfr)
        pn = max(pn, 1e-14)
        if abs(pn - p) <= 1e-15 * (pn + p):
            p = pn
            break
        p = pn
    fl, _ = _fK(p, rl, pl, gamma)
    fr, _ = _fK(p, rr, pr, gamma)
    u = 0.5 * (ul + ur) + 0.5 * (fr - fl)
    return p, u


def sample(left, right, gamma, xi):
    """Primitive solution (rho, u, p) at the similarity coordinates xi = (x - x0)/t."""
    rl, ul, pl = left
    rr, ur, pr = right
    ps, us = star_state(left, right, gamma)
    al, ar = np.sqrt(gamma * pl / rl), np.sqrt(gamma * pr / rr)
    g1 = (gamma - 1.0) / (gamma + 1.0)
    xi = np.asarray(xi, dtype=np.float64)
    rho = np.empty_like(xi)
    u = np.empty_like(xi)
    p = np.empty_like(xi)
    for n, s in enumerate(xi):
        if s <= us:  # left of the contact
            if ps > pl:  # left shock
                SL = ul - al * np.sqrt((gamma + 1) / (2 * gamma) * ps / pl + (gamma - 1) / (2 * gamma))
                if s <= SL:
                    rho[n], u[n], p[n] = rl, ul, pl
                else:
                    rho[n] = rl * (ps / pl + g1) / (g1 * ps / pl + 1.0)
                    u[n], p[n] = us, ps
            else:  # left rarefaction
                asl = al * (ps / pl) ** ((gamma - 1) / (2 * gamma))
                if s <= ul - al:
                    rho[n], u[n], p[n] = rl, ul, pl
                elif s >= us - asl:
                    rho[n] = rl * (ps / pl) ** (1.0 / gamma)
                    u[n], p[n] = us, ps
                else:
                    c = 2.0 / (gamma + 1) + g1 / al * (ul - s)
                    rho[n] = rl * c ** (2.0 / (gamma - 1))
                    u[n] = 2.0 / (gamma + 1) * (al + (gamma - 1) / 2 * ul + s)
                    p[n] = pl * c ** (2.0 * gamma / (gamma - 1))
        else:
            if ps > pr:  # right shock
                SR = ur + ar * np.sqrt((gamma + 1) / (2 * gamma) * ps / pr + (gamma - 1) / (2 * gamma))
                if s >= SR:
                    rho[n], u[n], p[n] = rr, ur, pr
                else:
                    rho[n] = rr * (ps / pr + g1) / (g1 * ps / pr + 1.0)
                    u[n], p[n] = us, ps
            else:  # right rarefaction
                asr = ar * (ps / pr) ** ((gamma - 1) / (2 * gamma))
                if s >= ur + ar:
                    rho[n], u[n], p[n] = rr, ur, pr
                elif s <= us + asr:
                    rho[n] = rr * (ps / pr) ** (1.0 / gamma)
                    u[n], p[n] = us, ps
                else:
                    c = 2.0 / (gamma + 1) - g1 / ar * (ur - s)
                    rho[n] = rr * c ** (2.0 / (gamma - 1))
                    u[n] = 2.0 / (gamma + 1) * (-ar + (gamma - 1) / 2 * ur + s)
                    p[n] = pr * c ** (2.0 * gamma / (gamma - 1))
    return rho, u, p

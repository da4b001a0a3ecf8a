"""ctypes binding of the CPU oracle (oracle/ox.h).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA package.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

CARTESIAN, SPHERICAL = 0, 1
BC_PERIODIC, BC_TRANSMISSIVE, BC_REFLECTING, BC_WEDGE = 0, 1, 2, 3
RIEMANN_HLL, RIEMANN_HLLC = 0, 1
LIM_NONE, LIM_MINMOD, LIM_VANLEER, LIM_VANALBADA, LIM_MC = 0, 1, 2, 3, 4
GRAV_NONE, GRAV_UNIFORM, GRAV_POINT_MASS, GRAV_SELF = 0, 1, 2, 3
SPACING_UNIFORM, SPACING_LOG, SPACING_CUSTOM = 0, 1, 2
CONSERVED, PRIMITIVE = 0, 1
OK, ERR_INVALID_ARG, ERR_ALLOC, ERR_NONPHYSICAL, ERR_UNSUPPORTED = 0, -1, -2, -4, -5


class OxConfig(C.Structure):
    _fields_ = [
        ("ndim", C.c_int), ("coords", C.c_int), ("n", C.c_int * 3),
        ("lo", C.c_double * 3), ("hi", C.c_double * 3), ("spacing", C.c_int * 3),
        ("faces", C.POINTER(C.c_double) * 3),
        ("bc_lo", C.c_int * 3), ("bc_hi", C.c_int * 3),
        ("eos", C.c_int), ("gamma", C.c_double),
        ("riemann", C.c_int), ("limiter", C.c_int), ("n_scalars", C.c_int),
        ("gravity", C.c_int), ("g", C.c_double * 3), ("GM", C.c_double),
        ("eos_R", C.c_double), ("eos_ar", C.c_double), ("G", C.c_double), ("emon_eps", C.c_double),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.c_int
        L.ox_create.argtypes = [C.POINTER(OxConfig), C.POINTER(vp)]
        L.ox_destroy.argtypes = [vp]
        L.ox_nvar.argtypes = [vp]
        L.ox_set_state.argtypes = [vp, dp, ip]
        L.ox_get_state.argtypes = [vp, dp, ip]
        L.ox_compute_dt.argtypes = [vp, C.c_double, dp]
        L.ox_step.argtypes = [vp, C.c_double]
        L.ox_cell_update.argtypes = [vp, ip, ip, ip, C.c_double, dp]
        L.ox_self_gravity.argtypes = [vp, ip, C.POINTER(C.c_double)]
        L.ox_riemann_flux.argtypes = [ip, C.c_double, ip, ip, ip, dp, dp, dp]
        for f in (L.ox_eos_pressure, L.ox_eos_energy, L.ox_eos_sound_speed):
            f.argtypes = [ip] + [C.c_double] * 5
            f.restype = C.c_double
        L.ox_physical_flux.argtypes = [C.c_double, ip, ip, ip, dp, dp]
        L.ox_limiter.argtypes = [ip, C.c_double, C.c_double]
        L.ox_limiter.restype = C.c_double
        L.ox_cell_geometry.argtypes = [vp, ip, ip, ip, dp, dp, dp]
        L.ox_faces.argtypes = [vp, ip, dp]
        L.ox_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def make_config(spec: dict) -> tuple:
    """Translate a plain-dict problem description (see paper_2503_04428_b200/workloads.py)
    into an OxConfig.  Returns (config, keepalive)."""
    cfg = OxConfig()
    ndim = int(spec["ndim"])
    cfg.ndim = ndim
    cfg.coords = int(spec.get("coords", CARTESIAN))
    keep = []
    n = list(spec["n"]) + [1] * (3 - len(spec["n"]))
    lo = list(spec.get("lo", [0.0] * 3)) + [0.0] * 3
    hi = list(spec.get("hi", [0.0] * 3)) + [0.0] * 3
    spacing = list(spec.get("spacing", [0] * 3)) + [0] * 3
    faces = list(spec.get("faces", [None] * 3)) + [None] * 3
    bc_lo = list(spec.get("bc_lo", [0] * 3)) + [0] * 3
    bc_hi = list(spec.get("bc_hi", [0] * 3)) + [0] * 3
    for d in range(3):
        cfg.n[d] = int(n[d])
        cfg.lo[d] = float(lo[d])
        cfg.hi[d] = float(hi[d])
        cfg.spacing[d] = int(spacing[d])
        cfg.bc_lo[d] = int(bc_lo[d])
        cfg.bc_hi[d] = int(bc_hi[d])
        if faces[d] is not None:
            arr = np.ascontiguousarray(faces[d], dtype=np.float64)
            keep.append(arr)
            cfg.faces[d] = _dptr(arr)
            cfg.spacing[d] = SPACING_CUSTOM
    cfg.eos = 0
    cfg.gamma = float(spec["gamma"])
    cfg.eos = int(spec.get("eos", 0))
    cfg.eos_R = float(spec.get("eos_R", 0.0))
    cfg.eos_ar = float(spec.get("eos_ar", 0.0))
    cfg.G = float(spec.get("G", 0.0))
    cfg.emon_eps = float(spec.get("emon_eps", 0.0))
    cfg.riemann = int(spec.get("riemann", RIEMANN_HLLC))
    cfg.limiter = int(spec.get("limiter", LIM_MINMOD))
    cfg.n_scalars = int(spec.get("n_scalars", 0))
    cfg.gravity = int(spec.get("gravity", GRAV_NONE))
    g = list(spec.get("g", [0.0] * 3)) + [0.0] * 3
    for d in range(3):
        cfg.g[d] = float(g[d])
    cfg.GM = float(spec.get("GM", 0.0))
    return cfg, keep


class OracleError(RuntimeError):
    def __init__(self, code, what):
        super().__init__(f"oracle {what} failed with code {code}")
        self.code = code


class Oracle:
    """The five calls of the boundary (create / set_state / compute_dt / step / get_state) on the CPU."""

    def __init__(self, spec: dict):
        self._L = lib()
        cfg, keep = make_config(spec)
        self._h = C.c_void_p()
        rc = self._L.ox_create(C.byref(cfg), C.byref(self._h))
        if rc != OK:
            raise OracleError(rc, "ox_create")
        self.ndim = cfg.ndim
        self.n = tuple(cfg.n)
        self.nvar = self._L.ox_nvar(self._h)
        self.shape = (self.nvar, self.n[2], self.n[1], self.n[0])

    def close(self):
        if self._h:
            self._L.ox_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_state(self, data: np.ndarray, form: int = CONSERVED):
        a = np.ascontiguousarray(data, dtype=np.float64)
        assert a.size == int(np.prod(self.shape)), (a.shape, self.shape)
        rc = self._L.ox_set_state(self._h, _dptr(a), form)
        if rc != OK:
            raise OracleError(rc, "ox_set_state")

    def get_state(self, form: int = CONSERVED) -> np.ndarray:
        out = np.empty(self.shape, dtype=np.float64)
        rc = self._L.ox_get_state(self._h, _dptr(out), form)
        if rc != OK:
            raise OracleError(rc, "ox_get_state")
        return out

    def compute_dt(self, cfl: float) -> float:
        dt = C.c_double()
        rc = self._L.ox_compute_dt(self._h, cfl, C.byref(dt))
        if rc != OK:
            raise OracleError(rc, "ox_compute_dt")
        return dt.value

    def step(self, dt: float):
        rc = self._L.ox_step(self._h, dt)
        if rc != OK:
            raise OracleError(rc, "ox_step")

    def cell_update(self, i: int, j: int, k: int, dt: float) -> np.ndarray:
        out = np.empty(self.nvar, dtype=np.float64)
        rc = self._L.ox_cell_update(self._h, i, j, k, dt, _dptr(out))
        if rc != OK:
            raise OracleError(rc, "ox_cell_update")
        return out

    def self_gravity(self, i: int) -> float:
        g = C.c_double()
        rc = self._L.ox_self_gravity(self._h, i, C.byref(g))
        if rc != OK:
            raise OracleError(rc, "ox_self_gravity")
        return g.value

    def cell_geometry(self, i, j, k):
        dV = C.c_double()
        dS = np.empty(6)
        xc = np.empty(3)
        rc = self._L.ox_cell_geometry(self._h, i, j, k, C.byref(dV), _dptr(dS), _dptr(xc))
        if rc != OK:
            raise OracleError(rc, "ox_cell_geometry")
        return dV.value, dS.reshape(3, 2), xc

    def faces(self, d: int) -> np.ndarray:
        ng = 2 if d < self.ndim else 0
        out = np.empty(self.n[d] + 1 + 2 * ng)
        rc = self._L.ox_faces(self._h, d, _dptr(out))
        if rc != OK:
            raise OracleError(rc, "ox_faces")
        return out


EOS_IDEAL, EOS_GAS_RADIATION = 0, 1


def eos_pressure(eos, gamma, R, ar, rho, e):
    return lib().ox_eos_pressure(eos, gamma, R, ar, rho, e)


def eos_energy(eos, gamma, R, ar, rho, P):
    return lib().ox_eos_energy(eos, gamma, R, ar, rho, P)


def eos_sound_speed(eos, gamma, R, ar, rho, P):
    return lib().ox_eos_sound_speed(eos, gamma, R, ar, rho, P)


def riemann_flux(riemann, gamma, ndim, ns, direction, UL, UR):
    UL = np.ascontiguousarray(UL, dtype=np.float64)
    UR = np.ascontiguousarray(UR, dtype=np.float64)
    F = np.empty_like(UL)
    rc = lib().ox_riemann_flux(riemann, gamma, ndim, ns, direction, _dptr(UL), _dptr(UR), _dptr(F))
    if rc != OK:
        raise OracleError(rc, "ox_riemann_flux")
    return F


def physical_flux(gamma, ndim, ns, direction, U):
    U = np.ascontiguousarray(U, dtype=np.float64)
    F = np.empty_like(U)
    rc = lib().ox_physical_flux(gamma, ndim, ns, direction, _dptr(U), _dptr(F))
    if rc != OK:
        raise OracleError(rc, "ox_physical_flux")
    return F


def limiter(lim, a, b):
    return lib().ox_limiter(lim, float(a), float(b))


def num_threads():
    return lib().ox_num_threads()

"""Thin ctypes binding over the C ABI of include/hx.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels of libhx.so; this module converts Python
arguments to pointers and sizes.  If libhx.so is missing it is built with nvcc (in-tree); if that
fails, or no CUDA device is present when a handle is created, the call raises -- there is no CPU
fallback and the CPU oracle is never imported from here.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

OK, ERR_INVALID_ARG, ERR_ALLOC, ERR_CUDA, ERR_NONPHYSICAL, ERR_UNSUPPORTED = 0, -1, -2, -3, -4, -5
CARTESIAN, SPHERICAL = 0, 1
BC_PERIODIC, BC_TRANSMISSIVE, BC_REFLECTING, BC_WEDGE = 0, 1, 2, 3
EOS_IDEAL, EOS_GAS_RADIATION = 0, 1
RIEMANN_HLL, RIEMANN_HLLC = 0, 1
LIM_NONE, LIM_MINMOD, LIM_VANLEER, LIM_VANALBADA, LIM_MC = 0, 1, 2, 3, 4
GRAV_NONE, GRAV_UNIFORM, GRAV_POINT_MASS, GRAV_SELF = 0, 1, 2, 3
SPACING_UNIFORM, SPACING_LOG, SPACING_CUSTOM = 0, 1, 2
HOST, DEVICE = 0, 1
CONSERVED, PRIMITIVE = 0, 1
OPT_KERNEL, OPT_TIMING, OPT_ASYNC_HOST = 0, 1, 2
KERNEL_AUTO, KERNEL_GENERIC, KERNEL_TILED = 0, 1, 2

EXPORTS = ["hx_create", "hx_destroy", "hx_set_stream", "hx_set_option", "hx_set_state", "hx_get_state",
           "hx_compute_dt", "hx_step", "hx_nvar", "hx_launch_count", "hx_kernel_time", "hx_step_kernel_name", "hx_last_error",
           "hx_version", "hx_probe_fp64", "hx_config_size", "hx_sync", "hx_self_gravity_table", "hx_self_gravity_noalloc", "hx_noalloc_error"]
NOALLOC_MAX_N0, NOALLOC_MAX_ANGULAR = 2048, 4096


class HxConfig(C.Structure):
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


class HxError(RuntimeError):
    def __init__(self, code, what, detail=""):
        super().__init__(f"{what} failed with code {code}" + (f": {detail}" if detail else ""))
        self.code = code


_lib = None


def lib_path():
    return _build.LIB


def lib():
    """Load libhx.so (building it in-tree first if needed).  Raises if it cannot be had."""
    global _lib
    if _lib is None:
        path = _build.ensure()
        if not os.path.exists(path):
            raise RuntimeError("libhx.so is missing and could not be built; the CUDA path has no fallback")
        L = C.CDLL(path)
        vp, dp = C.c_void_p, C.c_void_p
        L.hx_create.argtypes = [C.POINTER(HxConfig), C.POINTER(vp)]
        L.hx_destroy.argtypes = [vp]
        L.hx_set_stream.argtypes = [vp, vp]
        L.hx_set_option.argtypes = [vp, C.c_int, C.c_int]
        L.hx_set_state.argtypes = [vp, dp, C.c_int, C.c_int]
        L.hx_get_state.argtypes = [vp, dp, C.c_int, C.c_int]
        L.hx_compute_dt.argtypes = [vp, C.c_double, C.POINTER(C.c_double)]
        L.hx_step.argtypes = [vp, C.c_double]
        L.hx_sync.argtypes = [vp]
        L.hx_self_gravity_table.argtypes = [vp, dp, C.c_int]
        L.hx_self_gravity_noalloc.argtypes = [dp, dp, dp, dp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, dp, vp]
        L.hx_noalloc_error.restype = C.c_char_p
        L.hx_nvar.argtypes = [vp]
        L.hx_launch_count.argtypes = [vp]
        L.hx_launch_count.restype = C.c_longlong
        L.hx_kernel_time.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        L.hx_step_kernel_name.argtypes = [vp]
        L.hx_step_kernel_name.restype = C.c_char_p
        L.hx_last_error.argtypes = [vp]
        L.hx_last_error.restype = C.c_char_p
        L.hx_version.restype = C.c_char_p
        L.hx_probe_fp64.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double)]
        # ABI handshake: a stale libhx.so (or a stale binding) with another hx_config layout must not be used
        if not hasattr(L, "hx_config_size") or L.hx_config_size() != C.sizeof(HxConfig):
            have = L.hx_config_size() if hasattr(L, "hx_config_size") else "unknown"
            raise RuntimeError(f"{path}: hx_config is {have} bytes in the library but {C.sizeof(HxConfig)} in this binding; "
                               "rebuild with `python paper_2503_04428_b200/build.py --force`")
        _lib = L
    return _lib


def make_config(spec: dict):
    """Plain-dict problem description (workloads.py) -> HxConfig.  Returns (config, keepalive)."""
    cfg = HxConfig()
    cfg.ndim = int(spec["ndim"])
    cfg.coords = int(spec.get("coords", CARTESIAN))
    keep = []

    def three(key, fill):
        v = list(spec.get(key, []))
        return v + [fill] * (3 - len(v))
    n, lo, hi = three("n", 1), three("lo", 0.0), three("hi", 0.0)
    spacing, faces = three("spacing", 0), three("faces", None)
    bc_lo, bc_hi, g = three("bc_lo", 0), three("bc_hi", 0), three("g", 0.0)
    for d in range(3):
        cfg.n[d], cfg.lo[d], cfg.hi[d] = int(n[d]), float(lo[d]), float(hi[d])
        cfg.spacing[d], cfg.bc_lo[d], cfg.bc_hi[d], cfg.g[d] = int(spacing[d]), int(bc_lo[d]), int(bc_hi[d]), float(g[d])
        if faces[d] is not None:
            arr = np.ascontiguousarray(faces[d], dtype=np.float64)
            keep.append(arr)
            cfg.faces[d] = arr.ctypes.data_as(C.POINTER(C.c_double))
            cfg.spacing[d] = SPACING_CUSTOM
    cfg.eos = int(spec.get("eos", EOS_IDEAL))
    cfg.eos_R = float(spec.get("eos_R", 0.0))
    cfg.eos_ar = float(spec.get("eos_ar", 0.0))
    cfg.G = float(spec.get("G", 0.0))
    cfg.emon_eps = float(spec.get("emon_eps", 0.0))
    cfg.gamma = float(spec["gamma"])
    cfg.riemann = int(spec.get("riemann", RIEMANN_HLLC))
    cfg.limiter = int(spec.get("limiter", LIM_MINMOD))
    cfg.n_scalars = int(spec.get("n_scalars", 0))
    cfg.gravity = int(spec.get("gravity", GRAV_NONE))
    cfg.GM = float(spec.get("GM", 0.0))
    return cfg, keep


def _pointer(buf):
    """(address, mem_space, element count) of a numpy array (host) or a CUDA torch tensor (device)."""
    if isinstance(buf, np.ndarray):
        if buf.dtype != np.float64 or not buf.flags["C_CONTIGUOUS"]:
            raise TypeError("host buffers must be C-contiguous float64 numpy arrays")
        return buf.ctypes.data, HOST, buf.size
    if hasattr(buf, "data_ptr"):   # torch tensor
        import torch
        if buf.dtype != torch.float64 or not buf.is_contiguous():
            raise TypeError("tensors must be contiguous float64")
        return buf.data_ptr(), (DEVICE if buf.is_cuda else HOST), buf.numel()
    raise TypeError(f"unsupported buffer type {type(buf)}")


class Hydro:
    """One hx_handle.  Methods carry the names of the C calls without the hx_ prefix."""

    def __init__(self, spec: dict, stream=None):
        self._L = lib()
        cfg, _keep = make_config(spec)
        self._h = C.c_void_p()
        rc = self._L.hx_create(C.byref(cfg), C.byref(self._h))
        if rc != OK:
            raise HxError(rc, "hx_create", "no CUDA device" if rc == ERR_CUDA else "")
        self.ndim = cfg.ndim
        self.n = tuple(cfg.n)
        self.nvar = self._L.hx_nvar(self._h)
        self.shape = (self.nvar, self.n[2], self.n[1], self.n[0])
        self.size = int(np.prod(self.shape))
        if stream is not None:
            self.set_stream(stream)

    def _check(self, rc, what):
        if rc != OK:
            raise HxError(rc, what, self._L.hx_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._L.hx_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_stream(self, stream):
        ptr = stream if isinstance(stream, int) else getattr(stream, "cuda_stream", 0)
        self._check(self._L.hx_set_stream(self._h, C.c_void_p(ptr)), "hx_set_stream")

    def set_option(self, option, value):
        self._check(self._L.hx_set_option(self._h, option, value), "hx_set_option")

    def set_state(self, data, form=CONSERVED):
        ptr, space, count = _pointer(data)
        if count != self.size:
            raise ValueError(f"state buffer has {count} elements, expected {self.size}")
        self._check(self._L.hx_set_state(self._h, C.c_void_p(ptr), space, form), "hx_set_state")

    def get_state(self, out=None, form=CONSERVED):
        if out is None:
            out = np.empty(self.shape, dtype=np.float64)
        ptr, space, count = _pointer(out)
        if count != self.size:
            raise ValueError(f"state buffer has {count} elements, expected {self.size}")
        self._check(self._L.hx_get_state(self._h, C.c_void_p(ptr), space, form), "hx_get_state")
        return out

    def compute_dt(self, cfl: float) -> float:
        dt = C.c_double()
        self._check(self._L.hx_compute_dt(self._h, cfl, C.byref(dt)), "hx_compute_dt")
        return dt.value

    def step(self, dt: float):
        self._check(self._L.hx_step(self._h, dt), "hx_step")

    def sync(self):
        self._check(self._L.hx_sync(self._h), "hx_sync")

    def self_gravity_table(self):
        """HX_GRAV_SELF handles: the n[0] interior radial accelerations g_r(r_c,i) of the current state, through the handle's
        (cudaMalloc'ed) scratch -- the path hx_step uses."""
        out = np.empty(self.n[0], dtype=np.float64)
        self._check(self._L.hx_self_gravity_table(self._h, C.c_void_p(out.ctypes.data), HOST), "hx_self_gravity_table")
        return out

    def kernel_time(self):
        """(total ms, launches) of the step kernel alone, measured with CUDA events (OPT_TIMING on)."""
        ms, cnt = C.c_double(), C.c_longlong()
        self._check(self._L.hx_kernel_time(self._h, C.byref(ms), C.byref(cnt)), "hx_kernel_time")
        return ms.value, cnt.value

    @property
    def launch_count(self) -> int:
        return int(self._L.hx_launch_count(self._h))

    @property
    def step_kernel(self) -> str:
        return self._L.hx_step_kernel_name(self._h).decode()


def self_gravity_noalloc(rho, faces_r, faces_theta, faces_phi, GM, G, g, stream=None):
    """hx_self_gravity_noalloc: the self-gravity refresh of Eq. 4 with no device allocation (scratch in a static __device__
    array of the library).  All arrays are float64 CUDA tensors: rho [n2][n1][n0], the three face arrays, g [n0] (output).
    Asynchronous on `stream` (default: the legacy default stream).  Sizes beyond NOALLOC_MAX_N0 / NOALLOC_MAX_ANGULAR raise
    HxError(ERR_UNSUPPORTED)."""
    n2, n1, n0 = (int(x) for x in rho.shape)
    ptrs = []
    for name, buf, count in (("rho", rho, n0 * n1 * n2), ("faces_r", faces_r, n0 + 1), ("faces_theta", faces_theta, n1 + 1),
                             ("faces_phi", faces_phi, n2 + 1), ("g", g, n0)):
        ptr, space, have = _pointer(buf)
        if space != DEVICE:
            raise TypeError(f"{name} must be a CUDA tensor")
        if have != count:
            raise ValueError(f"{name} has {have} elements, expected {count}")
        ptrs.append(C.c_void_p(ptr))
    sp = 0 if stream is None else (stream if isinstance(stream, int) else getattr(stream, "cuda_stream", 0))
    L = lib()
    rc = L.hx_self_gravity_noalloc(ptrs[0], ptrs[1], ptrs[2], ptrs[3], n0, n1, n2, float(GM), float(G), ptrs[4], C.c_void_p(sp))
    if rc != OK:
        raise HxError(rc, "hx_self_gravity_noalloc", L.hx_noalloc_error().decode())


def probe_fp64():
    """(measured FP64 FMA throughput in TFLOP/s, dependent-DFMA latency in cycles) of the current GPU."""
    tf, lat = C.c_double(), C.c_double()
    rc = lib().hx_probe_fp64(C.byref(tf), C.byref(lat))
    if rc != OK:
        raise HxError(rc, "hx_probe_fp64")
    return tf.value, lat.value


def version() -> str:
    return lib().hx_version().decode()

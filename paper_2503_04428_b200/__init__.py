"""hx: a B200-native fp64 Godunov finite-volume hydro step (HERACLES++ hot path, arxiv 2503.04428).

`paper_2503_04428_b200.hx` is the thin ctypes binding over the C ABI of include/hx.h (loads
csrc/libhx.so, fails loudly if it is missing); `paper_2503_04428_b200.workloads` generates
the seeded synthetic inputs.  Nothing here falls back to a CPU implementation.
"""
__all__ = ["hx", "workloads"]

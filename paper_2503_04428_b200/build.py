"""Build the CUDA library IN-TREE: paper_2503_04428_b200/libhx.so (sm_100a only).

nvcc cross-compiles without a GPU; the .so travels to the GPU box with the repo snapshot.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
# HX_LIBRARY: load (and build into) another file, e.g. an A/B variant built with other -D flags
LIB = os.environ.get("HX_LIBRARY") or os.path.join(HERE, "libhx.so")
SOURCES = ["hx_host.cu", "hx_aux.cu", "hx_step_generic.cu", "hx_probe.cu", "hx_noalloc.cu",
           "hx_step_tile2.cu", "hx_step_tile2_nv5.cu", "hx_step_tile2_nv6.cu", "hx_step_tile2_nv7.cu", "hx_step_tile2_nv9.cu", "hx_step_tile2_nv9_rad.cu", "hx_step_tile2d.cu",
           "hx_step_tile2_nv8.cu", "hx_step_tile2_nv10.cu", "hx_step_tile2_nv11.cu", "hx_step_tile2_nv5_rad.cu", "hx_step_tile2_nv6_rad.cu",
           "hx_step_tile2_nv7_rad.cu", "hx_step_tile2_nv8_rad.cu", "hx_step_tile2_nv10_rad.cu", "hx_step_tile2_nv11_rad.cu"] + \
          ["hx_step_tile2_nv%d_emon.cu" % nv for nv in range(5, 12)] + ["hx_step_tile2_nv%d_rad_emon.cu" % nv for nv in range(5, 12)]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"]


def _deps():
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(ROOT, "include", "hx.h")]
    return max(os.path.getmtime(p) for p in deps)


def build(force: bool = False, verbose: bool = False, extra_flags=(), lib: str = None, objdir: str = None) -> str:
    """extra_flags / lib / objdir: variant builds (other -D flags into another .so, objects kept apart)."""
    lib = lib or LIB
    objdir = objdir or CSRC
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= _deps():
        return lib
    os.makedirs(objdir, exist_ok=True)
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    # one nvcc per translation unit, at most `jobs` at a time (HX_BUILD_JOBS, default: the cores of this box): 35 compilers at once
    # need tens of GB of memory; the heaviest units (gas + radiation EOS builds) go first so that they do not end up alone at the tail
    jobs = max(1, int(os.environ.get("HX_BUILD_JOBS", "0")) or (os.cpu_count() or 4))
    order = sorted(SOURCES, key=lambda f: (0 if "_rad" in f else 1 if "tile2" in f else 2))
    objs = [os.path.join(objdir, src.replace(".cu", ".o")) for src in SOURCES]
    pending, running, failed = list(order), [], None
    while (pending or running) and failed is None:
        while pending and len(running) < jobs:
            src = pending.pop(0)
            obj = os.path.join(objdir, src.replace(".cu", ".o"))
            cmd = [nvcc] + NVCC_FLAGS + list(extra_flags) + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, src), "-o", obj]
            running.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        src, p = running.pop(0)                 # wait for the oldest one (they finish roughly in order)
        out, _ = p.communicate()
        if verbose or p.returncode != 0:
            sys.stderr.write(out)
        if p.returncode != 0:
            failed = src
    for _, p in running:
        p.kill()
    if failed is not None:
        raise RuntimeError(f"nvcc failed on {failed}")
    cmd = [nvcc, "-shared", "-o", lib] + objs + ["-lcudart", "-lcuda"]
    subprocess.run(cmd, check=True)
    return lib


def ensure() -> str:
    """Build only if the library is missing (the GPU box gets the .so with the repo snapshot;
    file times there are not reliable enough for a staleness check)."""
    return LIB if os.path.exists(LIB) else build(force=True)


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))

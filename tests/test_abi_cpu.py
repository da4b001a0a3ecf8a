"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol include/hx.h
declares; argument validation that needs no GPU; no CPU fallback."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2503_04428_b200 import hx, workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "hx.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hx_[a-z0-9_]+)\s*\(", text)))


def test_library_loads_and_exports_every_declared_symbol():
    L = hx.lib()
    names = declared_functions()
    assert set(names) == set(hx.EXPORTS), (names, hx.EXPORTS)
    for name in names:
        assert hasattr(L, name), name
    assert b"sm_100a" in L.hx_version()
    assert L.hx_config_size() == C.sizeof(hx.HxConfig)      # the handshake hx.lib() enforces


def test_config_struct_matches_header_layout():
    # 3 ints, 6 doubles, 3 ints, 3 pointers, 6 ints, int + double, 3 ints, int, 3 doubles, double, 2 doubles (EOS constants)
    assert C.sizeof(hx.HxConfig) == 232
    assert hx.HxConfig.faces.offset == 88 and hx.HxConfig.gamma.offset == 144 and hx.HxConfig.GM.offset == 192
    assert hx.HxConfig.eos_R.offset == 200 and hx.HxConfig.eos_ar.offset == 208 and hx.HxConfig.G.offset == 216 and hx.HxConfig.emon_eps.offset == 224


def test_invalid_arguments_rejected_without_gpu():
    L = hx.lib()
    out = C.c_void_p()
    assert L.hx_create(None, C.byref(out)) == hx.ERR_INVALID_ARG
    spec, _ = wl.sod_1d(16)
    for key, val in (("gamma", 1.0), ("ndim", 4), ("limiter", 9), ("riemann", 5), ("n_scalars", 40), ("eos", 1)):   # eos 1 (gas + radiation) without its constants
        bad = dict(spec)
        bad[key] = val
        cfg, keep = hx.make_config(bad)
        assert L.hx_create(C.byref(cfg), C.byref(out)) == hx.ERR_INVALID_ARG, key
        assert not out.value
    bad = dict(spec, eos=2)                          # unknown equation of state
    cfg, keep = hx.make_config(bad)
    assert L.hx_create(C.byref(cfg), C.byref(out)) == hx.ERR_UNSUPPORTED
    bad = dict(spec)
    bad["bc_lo"] = [hx.BC_PERIODIC, 0, 0]          # periodic on one side only
    cfg, keep = hx.make_config(bad)
    assert L.hx_create(C.byref(cfg), C.byref(out)) == hx.ERR_INVALID_ARG
    bad = dict(spec)
    bad["faces"] = [np.array(spec["faces"][0])[::-1].copy(), None, None]   # decreasing faces
    cfg, keep = hx.make_config(bad)
    assert L.hx_create(C.byref(cfg), C.byref(out)) == hx.ERR_INVALID_ARG
    assert L.hx_destroy(None) == hx.OK
    assert L.hx_step(None, 0.1) == hx.ERR_INVALID_ARG


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    spec, _ = wl.sod_1d(16)
    with pytest.raises(hx.HxError) as e:
        hx.Hydro(spec)
    assert e.value.code == hx.ERR_CUDA


def test_product_path_never_imports_the_oracle():
    """Neither side includes, imports or links the other (comments may name the other side)."""
    inc = re.compile(r'^\s*#\s*include\s*[<"]([^>"]+)[>"]', re.M)
    imp = re.compile(r"^\s*(?:from|import)\s+([\w\.]+)", re.M)
    pkg = os.path.join(ROOT, "paper_2503_04428_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if not f.endswith((".py", ".cu", ".cuh", ".h")):
                continue
            text = open(os.path.join(dirpath, f)).read()
            assert not [x for x in inc.findall(text) if "ox" in os.path.basename(x) or "oracle" in x], f
            if f.endswith(".py"):
                assert not [x for x in imp.findall(text) if x.split(".")[0] in ("oracle", "tests")], f
                assert "libox" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if not f.endswith((".py", ".cpp", ".h")):
            continue
        text = open(os.path.join(ROOT, "oracle", f)).read()
        assert not [x for x in inc.findall(text) if "hx" in os.path.basename(x) or "cuda" in x], f
        if f.endswith(".py"):
            assert not [x for x in imp.findall(text) if x.startswith("paper_2503_04428_b200")], f
            assert "libhx" not in text, f

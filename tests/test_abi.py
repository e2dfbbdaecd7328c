"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol include/nsgw.h declares;
the product binding never touches the oracle; without a GPU it fails loudly instead of falling back."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "nsgw.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(?:int|int64_t|void|const char\*)\s+\*?\s*((?:ns_|gw_|nsgw_)\w+)\s*\(", src)
    return sorted(set(names))


def test_header_symbols_exported():
    from paper_2509_04336_b200 import build, nsgw
    lib = ctypes.CDLL(build.build())
    declared = _declared()
    assert len(declared) >= 14
    for n in declared:
        assert hasattr(lib, n), n
    assert sorted(nsgw.EXPORTS) == declared


def test_product_does_not_import_oracle():
    imp = re.compile(r"^\s*(from|import)\s+\S*oracle|#include\s+\S*oracle|liboracle", re.M)
    pkg = os.path.join(ROOT, "paper_2509_04336_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not imp.search(open(os.path.join(dirpath, f)).read()), f
    # the oracle side may use the seeded INPUT generators (workloads.py holds none of the method's arithmetic) and nothing else
    back = re.compile(r"^\s*(from|import)\s+paper_2509_04336_b200(?!\s+import\s+workloads\b)|#include\s+\S*nsgw", re.M)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            assert not back.search(open(os.path.join(ROOT, "oracle", f)).read()), f
    wl = open(os.path.join(pkg, "workloads.py")).read()
    assert not re.search(r"^\s*(from|import)\s+(\.|paper_2509_04336_b200|torch|ctypes)", wl, re.M)   # inputs only: no binding, no library


def test_no_cpu_fallback():
    import torch
    from paper_2509_04336_b200 import nsgw, workloads as W
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    spec, smp, _ = W.config1()
    with pytest.raises(nsgw.NsgwError):
        nsgw.Handle(spec, smp)
    # the raw C call reports a CUDA error rather than computing anything
    cfg, _ = nsgw.make_config(spec, smp)
    h = ctypes.c_void_p(0)
    rc = nsgw.lib().ns_init(ctypes.byref(h), ctypes.byref(cfg), None, None, None, ctypes.c_uint64(1), None)
    assert rc == -2 and not h.value
    assert b"no CUDA device" in nsgw.lib().ns_last_error(None)


def test_argument_validation_without_gpu():
    from paper_2509_04336_b200 import nsgw, workloads as W
    spec, smp, _ = W.config1()
    bad = dict(smp, n_delete=smp["n_live"] - 1)
    cfg, _ = nsgw.make_config(spec, bad)
    h = ctypes.c_void_p(0)
    assert nsgw.lib().ns_init(ctypes.byref(h), ctypes.byref(cfg), None, None, None, ctypes.c_uint64(1), None) == -1
    cfg, _ = nsgw.make_config(dict(spec, like_kind=1), smp)      # GW kind with ndim = 4
    assert nsgw.lib().ns_init(ctypes.byref(h), ctypes.byref(cfg), None, None, None, ctypes.c_uint64(1), None) == -5
    cfg, _ = nsgw.make_config(spec, smp)
    cfg.struct_version = 7
    assert nsgw.lib().ns_init(ctypes.byref(h), ctypes.byref(cfg), None, None, None, ctypes.c_uint64(1), None) == -1

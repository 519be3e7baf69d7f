"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/rt.h declares; host-only entry points work; compute entry points fail loudly without a GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "rt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rt_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_exported():
    import paper_1410_0763_b200 as rt
    L = rt.load_library()
    names = declared_symbols()
    assert len(names) >= 12
    for n in names:
        assert hasattr(L, n), "librt.so does not export %s" % n
    assert sorted(rt.EXPORTED_SYMBOLS) == names


def test_library_is_in_tree_and_sm100a():
    import paper_1410_0763_b200.build as b
    assert os.path.exists(b.LIB) and b.LIB.startswith(ROOT)
    flags = " ".join(b.NVCC_FLAGS)
    assert "arch=compute_100a,code=sm_100a" in flags and "-lineinfo" in flags


def test_host_only_entry_points():
    import paper_1410_0763_b200 as rt
    d = rt.healpix_dirs(4)
    assert d.shape == (192, 3) and np.abs(np.linalg.norm(d, axis=1) - 1).max() < 1e-15
    L = rt.load_library()
    assert L.rt_strerror(0) == b"ok" and L.rt_strerror(-1) == b"invalid argument"
    assert L.rt_healpix_dirs(0, None) == -1
    assert L.rt_destroy(None) == 0


def test_no_cpu_fallback():
    """Without a CUDA device rt_create must fail with RT_ECUDA (never compute on the host)."""
    import torch
    import paper_1410_0763_b200 as rt
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(rt.RtError) as ei:
        rt.rt_create(8, 8, 8, 1, rt.healpix_dirs(1))
    assert ei.value.code == -3


def test_product_does_not_import_oracle():
    """The product path may not import, call, link or execute anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1410_0763_b200")
    bad = re.compile(r"import\s+oracle|from\s+oracle|from\s+\.+oracle|liboracle|\borc_[a-z]|oracle\.(c|py|h)\b")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not bad.search(txt), "%s references the oracle" % f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1410_0763_b200" not in txt and "librt" not in txt

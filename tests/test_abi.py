"""CPU-only checks of the boundary: libcbct.so loads, exports every symbol include/cbct.h declares,
validates arguments, and fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cb():
    import paper_1002_3675_b200 as cb
    from paper_1002_3675_b200 import build
    build.build()                      # nvcc cross-compiles without a GPU
    cb.load()
    return cb


def test_library_exports_every_declared_symbol(cb):
    hdr = open(os.path.join(ROOT, "include", "cbct.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(cbct_[a-z0-9_]+)\s*\(", hdr))
    assert {"cbct_geometry_create", "cbct_forward", "cbct_backproject", "cbct_tv_prox",
            "cbct_fbs_reconstruct"} <= declared
    from paper_1002_3675_b200.binding import SYMBOLS
    assert declared == set(SYMBOLS)
    lib = ctypes.CDLL(cb.lib_path())
    for name in declared:
        assert hasattr(lib, name), name


def test_sources_target_sm100a_only():
    from paper_1002_3675_b200 import build
    assert "arch=compute_100a,code=sm_100a" in build.FLAGS and "-lineinfo" in build.FLAGS
    assert len(build.sources()) >= 5


def test_argument_validation_and_no_cpu_fallback(cb):
    import torch
    ang = np.zeros(3)
    with pytest.raises(cb.CbctError) as e:
        cb.Geometry(1500, 1000, ang, 8, 8, 1, 1, 8, 8, 8, 1, 1, 1)           # sad >= sdd
    assert e.value.status == 1
    with pytest.raises(cb.CbctError) as e:
        cb.Geometry(1000, 1500, ang, 8, 8, 1, 1, 0, 8, 8, 1, 1, 1)           # nx = 0
    assert e.value.status == 1
    with pytest.raises(cb.CbctError) as e:
        cb.Geometry(100, 1500, ang, 8, 8, 1, 1, 256, 256, 8, 1, 1, 1)        # volume reaches the source
    assert e.value.status == 2
    if not torch.cuda.is_available():
        with pytest.raises(cb.CbctError) as e:
            cb.Geometry(1000, 1500, ang, 8, 8, 1, 1, 8, 8, 8, 1, 1, 1)
        assert e.value.status == 4 and "no CPU fallback" in str(e.value)
    assert cb.launch_count() >= 0


def test_product_does_not_import_the_oracle():
    """The product path may not route through oracle/ (or cbct_synth): grep the package sources."""
    pkg = os.path.join(ROOT, "paper_1002_3675_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), fn
                assert "liboracle" not in src and "cbct_oracle" not in src, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "paper_1002_3675_b200" not in src.replace("`paper_1002_3675_b200`", "").replace(
                "paper_1002_3675_b200/csrc", "") or fn == "__init__.py", fn
            assert "libcbct" not in src, fn

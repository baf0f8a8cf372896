"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/igr.h declares and
fails loudly (never falls back) when no GPU is present.  No compute calls."""
import ctypes as C
import os
import re

import pytest
import torch

from paper_2505_07392_b200 import build, igr

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return igr.lib()


def test_library_exports_every_declared_symbol(lib):
    header = open(os.path.join(ROOT, "include", "igr.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = sorted(set(re.findall(r"\b(igr_[a-z0-9_]+)\s*\(", header)))
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(igr.EXPORTS) == declared


def test_workspace_bytes_counts_the_fields(lib):
    opt = igr.Options()
    n = 64
    b32 = lib.igr_workspace_bytes(n, n, n, C.byref(opt))
    field = (n + 16) * (n + 6) * (n + 6) * 4
    assert 18 * field <= b32 <= 18 * field + (80 << 20)      # 10 q + 2 Sigma + b + 5 r, + staging
    opt.storage = igr.STORE_F16
    b16 = lib.igr_workspace_bytes(n, n, n, C.byref(opt))
    assert b16 < b32
    opt.fused = 1                                             # third state buffer, but r[5] is not resident
    opt.storage = igr.STORE_F32
    bf = lib.igr_workspace_bytes(n, n, n, C.byref(opt))
    assert 18 * field <= bf <= 18 * field + (80 << 20)       # 15 q + 2 Sigma + b, + staging
    opt.variant = igr.VARIANT_SIMPLE                          # the simple kernels always run the unfused rows
    assert lib.igr_workspace_bytes(n, n, n, C.byref(opt)) >= 23 * field
    assert lib.igr_workspace_bytes(0, n, n, C.byref(opt)) == 0


def test_create_validates_arguments_and_never_falls_back(lib):
    bc, _ = igr.make_bc((0,) * 6)
    h = C.c_void_p()
    assert lib.igr_create(8, 8, 8, 0.1, 1.4, 0.1, 4, 5, C.byref(bc), C.byref(h)) == igr.ERR_ARG
    assert lib.igr_create(8, 8, 8, 0.1, 1.0, 0.1, 5, 5, C.byref(bc), C.byref(h)) == igr.ERR_ARG
    assert lib.igr_create(8, 8, 0, 0.1, 1.4, 0.1, 5, 5, C.byref(bc), C.byref(h)) == igr.ERR_ARG
    bad, _ = igr.make_bc((0, 1, 0, 0, 0, 0))
    assert lib.igr_create(8, 8, 8, 0.1, 1.4, 0.1, 5, 5, C.byref(bad), C.byref(h)) == igr.ERR_BC
    if not torch.cuda.is_available():
        assert lib.igr_create(8, 8, 8, 0.1, 1.4, 0.1, 5, 5, C.byref(bc), C.byref(h)) == igr.ERR_CUDA
        assert not h.value
        with pytest.raises(igr.IgrError):
            igr.Solver(8, 8, 8, 0.1, 1.4, 0.1)
    assert lib.igr_step(None, 0.1) == igr.ERR_ARG
    assert lib.igr_max_wavespeed(None, None) == igr.ERR_ARG

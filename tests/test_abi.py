"""CPU-side checks of the boundary: the library builds/loads, exports every symbol include/b200sht.h declares,
validates arguments, and fails loudly (no CPU fallback).  No compute calls here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2311_14670_b200 import build, _lib
    build.build()
    return _lib.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "b200sht.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b([a-z0-9_]+)\s*\(", src)
    return sorted({n for n in names if n.startswith(("sht_", "s2_", "so3_"))})


def test_every_declared_symbol_is_exported_and_bound(lib):
    from paper_2311_14670_b200 import _lib
    decl = declared_symbols()
    assert len(decl) >= 25
    for name in decl:
        assert hasattr(lib, name), f"{name} declared in b200sht.h but not exported"
        assert name in _lib.SIGNATURES, f"{name} has no ctypes signature"
    assert sorted(_lib.SIGNATURES) == decl


def test_status_strings_and_argument_validation(lib):
    assert lib.sht_status_string(0) == b"SHT_OK"
    assert b"EINVAL" in lib.sht_status_string(1)
    h = C.c_void_p()
    assert lib.sht_plan_s2(C.byref(h), 0, 0, 0, 0, 0, 0) == 1          # L < 1
    assert lib.sht_plan_s2(C.byref(h), 8, 8, 0, 0, 0, 0) == 1          # |spin| >= L
    assert lib.sht_plan_s2(C.byref(h), 8, 2, 0, 0, 1, 0) == 1          # reality needs spin 0 (R15)
    assert lib.sht_plan_s2(C.byref(h), 8, 0, 7, 0, 0, 0) == 1          # unknown sampling
    assert lib.sht_plan_s2(C.byref(h), 8, 0, 1, 0, 0, 0) == 1          # HEALPix needs nside >= 1
    assert lib.sht_plan_so3_opts(C.byref(h), 8, 3, 1, 32) == 2                    # fp32 arrays: not with SHT_OPT_ADJOINT
    assert lib.sht_plan_s2_opts(C.byref(h), 8, 2, 0, 0, 0, 1, 1, 32) == 2
    assert lib.sht_plan_so3(C.byref(h), 8, 3, 7) == 1                  # unknown dtype
    assert lib.sht_plan_s2(C.byref(h), 8, 0, 0, 0, 0, 7) == 1          # unknown dtype
    assert lib.sht_plan_so3(C.byref(h), 8, 9, 0) == 1                  # N > L
    assert lib.sht_plan_s2(C.byref(h), 8, 0, 9, 0, 0, 0) == 1          # sampling codes are 0..4 (MW, HEALPix, MWSS, DH, GL)
    assert lib.sht_plan_s2_opts(C.byref(h), 8, 0, 0, 0, 0, 0, 1, 1 | 2) == 1      # SHT_OPT_FOLD_ON with SHT_OPT_FOLD_OFF
    assert lib.sht_plan_s2_opts(C.byref(h), 8, 0, 0, 0, 0, 0, 1, 4 | 128) == 1    # SHT_OPT_INVSYM with SHT_OPT_NO_INVSYM
    assert lib.sht_plan_s2_opts(C.byref(h), 8, 0, 0, 0, 0, 1, 1, 64) == 2         # precompute is fp64 only
    assert lib.sht_plan_s2_opts(C.byref(h), 8, 0, 0, 0, 0, 0, 1, 512 | 1024) == 1 # SHT_OPT_GRAPH with SHT_OPT_NO_GRAPH
    assert lib.sht_plan_set_shard(None, 0, 1) == 1
    assert lib.sht_peak(7, 10, None, None, None) == 1
    assert lib.sht_plan_workspace_bytes(None) == 0
    assert lib.s2_forward_plan(None, None, None, None) == 1


def test_band_limit_beyond_the_window_counter_range_is_refused(lib):
    """Eq. 27 start values below 2^-122900 do not fit the one-byte window counter; they must never be dropped silently.
    The range check runs on the host before any CUDA call, so it is testable without a GPU: MW plans are refused from L ~ 9100."""
    h = C.c_void_p()
    for L in (9300, 12000, 16384):
        assert lib.sht_plan_s2(C.byref(h), L, 0, 0, 0, 0, 0) == 2, L                # SHT_EUNSUPPORTED
        assert b"start values" in lib.sht_last_error()
    assert lib.sht_plan_s2(C.byref(h), 9300, 2, 3, 0, 0, 0) == 2                    # DH: same rings as the MW quadrature
    assert lib.sht_plan_so3(C.byref(h), 9300, 4, 0) == 2


def test_no_cpu_fallback_without_gpu(lib):
    """On a box without a GPU a plan cannot be created: the call must return an error code, never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = C.c_void_p()
    rc = lib.sht_plan_s2(C.byref(h), 16, 0, 0, 0, 0, 0)
    assert rc in (4, 5) and lib.sht_last_error() != b""
    from paper_2311_14670_b200 import api
    with pytest.raises(Exception):
        api.Plan(16, 0)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2311_14670_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".h", ".cuh")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "sht_oracle" not in txt, fn
    otxt = open(os.path.join(ROOT, "oracle", "sht_oracle.cpp")).read() + open(os.path.join(ROOT, "oracle", "oracle.py")).read()
    assert "paper_2311_14670_b200" not in otxt.replace("paper_2311_14670_b200/csrc", "")

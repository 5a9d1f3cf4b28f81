"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol include/*.h
declare, validates arguments, and fails loudly (CAV_ECUDA, no CPU fallback) when there is no CUDA device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cav():
    from paper_0809_3098_b200 import binding
    return binding


def declared_symbols(headers=None):
    """every function any include/*.h declares (or only the given headers)"""
    inc = os.path.join(ROOT, "include")
    names = set()
    for h in sorted(headers or [f for f in os.listdir(inc) if f.endswith(".h")]):
        src = open(os.path.join(inc, h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(cav_[a-z_0-9]+)\s*\(", src))
    return sorted(names)


def test_cavity_h_is_the_methods_boundary_only():
    # SURVEY S8(b)'s calls plus the documented product additions; tuning / tracing / testing aids live in cavity_debug.h
    assert declared_symbols(["cavity.h"]) == sorted([
        "cav_create", "cav_destroy", "cav_set_fields", "cav_get_fields", "cav_step", "cav_step_async", "cav_sync", "cav_poisson",
        "cav_get_diag", "cav_set_sweep", "cav_step_res", "cav_run_to_steady", "cav_diag_noalloc", "cav_noalloc_max_n", "cav_strerror"])
    assert len(declared_symbols(["cavity_debug.h"])) == 10


def test_header_declares_the_north_star_calls():
    names = declared_symbols()
    for need in ("cav_create", "cav_step", "cav_poisson", "cav_get_fields", "cav_destroy", "cav_set_fields"):
        assert need in names


def test_library_exports_every_declared_symbol(cav):
    L = cav.lib()
    names = declared_symbols()
    assert sorted(cav.SYMBOLS) == names
    for n in names:
        assert getattr(L, n) is not None, n


def test_no_oracle_or_cpu_fallback_in_product():
    # the product package never imports or links the oracle
    pkg = os.path.join(ROOT, "paper_0809_3098_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "liboracle" not in text and "cavity_oracle" not in text, f


def test_strerror(cav):
    L = cav.lib()
    assert L.cav_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4, -99):
        assert len(L.cav_strerror(code)) > 0


def test_create_rejects_bad_arguments(cav):
    L = cav.lib()
    h = C.c_void_p()
    bad = [(1, 100.0, 0.01, 1.8, 10), (32, 0.0, 0.01, 1.8, 10), (32, -5.0, 0.01, 1.8, 10), (32, 100.0, 0.0, 1.8, 10),
           (32, 100.0, 0.01, 0.0, 10), (32, 100.0, 0.01, 2.0, 10), (32, 100.0, 0.01, 1.8, -1),
           (32, float("nan"), 0.01, 1.8, 10), (32, 100.0, float("inf"), 1.8, 10)]
    for args in bad:
        assert L.cav_create(C.byref(h), *args) == -1, args
        assert not h.value
    assert L.cav_create(None, 32, 100.0, 0.01, 1.8, 10) == -1


def test_null_context_is_rejected(cav):
    L = cav.lib()
    assert L.cav_step(None, 1) == -1
    assert L.cav_poisson(None, 1, None) == -1
    assert L.cav_get_fields(None, None, None) == -1
    assert L.cav_get_diag(None, None) == -1
    assert L.cav_launch_count(None) == 0
    L.cav_destroy(None)   # no-op


def test_create_without_gpu_fails_loudly(cav):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = C.c_void_p()
    assert cav.lib().cav_create(C.byref(h), 32, 100.0, 0.0156, 1.8, 20) == -3     # CAV_ECUDA
    assert not h.value
    with pytest.raises(cav.CavityError):
        cav.Cavity(32, 100.0, 0.0156, 1.8, 20)

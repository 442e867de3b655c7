"""CPU-side checks of the boundary: libplspec.so builds, loads and exports every symbol that
include/plspec.h declares; status strings; graceful failure without a device.  No compute."""
import ctypes
import os
import re

import pytest

from paper_2311_18737_b200 import binding as pl
from paper_2311_18737_b200 import build as plbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "plspec.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(plspec_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    plbuild.build()
    return pl.lib()


def test_header_and_binding_agree():
    assert declared_functions() == sorted(pl.EXPORTED_SYMBOLS)


def test_library_exports_every_declared_symbol(lib):
    raw = ctypes.CDLL(pl.LIB_PATH)
    for name in declared_functions():
        assert hasattr(raw, name), f"libplspec.so does not export {name}"


def test_strerror_and_version(lib):
    assert pl.strerror(pl.PLSPEC_OK) == "ok"
    for code in (pl.PLSPEC_ERR_INVALID_ARG, pl.PLSPEC_ERR_ALLOC, pl.PLSPEC_ERR_CUDA, pl.PLSPEC_ERR_UNSUPPORTED, -99):
        assert isinstance(pl.strerror(code), str) and pl.strerror(code)
    assert "plspec" in pl.plspec_version()


def test_no_silent_cpu_fallback(lib):
    """Without a CUDA device create must fail with an error code -- never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = ctypes.c_void_p(123)
    rc = lib.plspec_create(1024, 1024, 4, 0, 1, 0, 0, ctypes.byref(h))
    assert rc in (pl.PLSPEC_ERR_CUDA, pl.PLSPEC_ERR_UNSUPPORTED) and not h.value
    rc = lib.plspec_create(1000, 1024, 4, 0, 1, 0, 0, ctypes.byref(h))
    assert rc == pl.PLSPEC_ERR_INVALID_ARG          # argument checks come first, device or not
    assert lib.plspec_accumulate(None, None, None, 1, None) == pl.PLSPEC_ERR_INVALID_ARG
    assert lib.plspec_finalize(None, None) == pl.PLSPEC_ERR_INVALID_ARG


def test_binding_has_no_compute():
    """The binding marshals arguments only: no numpy/torch arithmetic on data inside it."""
    src = open(os.path.join(ROOT, "paper_2311_18737_b200", "binding.py")).read()
    for banned in ("np.fft", "torch.fft", "np.abs", "np.conj", "oracle"):
        assert banned not in src.split('"""', 2)[2], banned


def test_header_and_binding_constants_agree():
    """Every PLSPEC_* enumerator of include/plspec.h has the same value in the binding."""
    src = open(os.path.join(ROOT, "include", "plspec.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    consts = dict((k, int(v)) for k, v in re.findall(r"\b(PLSPEC_[A-Z0-9_]+)\s*=\s*(-?\d+)", src))
    assert {"PLSPEC_OK", "PLSPEC_SC16", "PLSPEC_OPT_SPLIT", "PLSPEC_OPT_SHARED_CODE"} <= set(consts)
    for name, value in consts.items():
        if hasattr(pl, name):
            assert getattr(pl, name) == value, name
    for name in ("PLSPEC_OPT_KERNEL", "PLSPEC_OPT_IPP_CHUNKS", "PLSPEC_OPT_H2D_BATCH", "PLSPEC_OPT_BPSK_PACK",
                 "PLSPEC_OPT_STAGE", "PLSPEC_OPT_SPLIT", "PLSPEC_OPT_SHARED_CODE"):
        assert getattr(pl, name) == consts[name], name


def test_handle_free_calls_check_their_arguments_before_touching_the_device(lib):
    """Argument errors of the diagnostic / product calls come first, with or without a GPU."""
    d = ctypes.c_double()
    vp = ctypes.c_void_p
    assert lib.plspec_diag_fp32_peak(2, 1, 1, ctypes.byref(d), ctypes.byref(d), None) == pl.PLSPEC_ERR_INVALID_ARG
    assert lib.plspec_diag_fp32_peak(1, 0, 1, ctypes.byref(d), ctypes.byref(d), None) == pl.PLSPEC_ERR_INVALID_ARG
    assert lib.plspec_diag_fp32_peak(1, 1, 1, None, ctypes.byref(d), None) == pl.PLSPEC_ERR_INVALID_ARG
    assert lib.plspec_diag_mem_bandwidth(9, 1 << 25, 8, 1, ctypes.byref(d), None) == pl.PLSPEC_ERR_INVALID_ARG
    assert lib.plspec_diag_mem_bandwidth(0, 1000, 8, 1, ctypes.byref(d), None) == pl.PLSPEC_ERR_INVALID_ARG
    assert lib.plspec_diag_mem_bandwidth(0, 1 << 25, 8, 1, None, None) == pl.PLSPEC_ERR_INVALID_ARG
    assert lib.plspec_finalize_products(None, None, None) == pl.PLSPEC_ERR_INVALID_ARG
    assert lib.plspec_profile(None, 4, 1024, 1, 1, 0, None, None, None, None, None, None) == pl.PLSPEC_ERR_INVALID_ARG
    assert lib.plspec_mean_spectrum(None, None, 4, 1024, 1, 0, None) == pl.PLSPEC_ERR_INVALID_ARG
    assert lib.plspec_profile_static(None, 4, 1024, 1, 1, 0, None, None, None, None, None, None) == pl.PLSPEC_ERR_INVALID_ARG
    one = ctypes.c_float()                              # size beyond the static workspace: refused before any CUDA call
    ptrs = [ctypes.cast(ctypes.byref(one), vp)] * 5
    assert lib.plspec_profile_static(ctypes.cast(ctypes.byref(one), vp), pl.STATIC_MAX_GATES + 1, 1024, 1, 1, 0, *ptrs,
                                     None) == pl.PLSPEC_ERR_INVALID_ARG
    assert lib.plspec_configure(None, pl.PLSPEC_OPT_SPLIT, 1) == pl.PLSPEC_ERR_INVALID_ARG
    assert lib.plspec_get_stats(None, None) == pl.PLSPEC_ERR_INVALID_ARG and lib.plspec_reset(None) == pl.PLSPEC_ERR_INVALID_ARG

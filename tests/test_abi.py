"""The C-ABI library builds for sm_100a without a GPU, loads, and exports every symbol include/mwax_corr.h
declares.  No compute call is made here."""
import ctypes
import os
import re

import pytest

from paper_2303_11557_b200 import corr

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "mwax_corr.h")


def _declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mwax_x?corr_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    syms = _declared_symbols()
    for s in ("mwax_corr_create", "mwax_corr_process", "mwax_corr_destroy", "mwax_xcorr_i8_create",
              "mwax_xcorr_i8_process", "mwax_xcorr_i8_destroy", "mwax_corr_process_batch", "mwax_corr_process_host"):
        assert s in syms


def test_library_builds_loads_and_exports_every_declared_symbol():
    path = corr.build()
    lib = ctypes.CDLL(path)
    for s in _declared_symbols():
        assert hasattr(lib, s), f"{s} declared in mwax_corr.h but not exported"


def test_strerror_and_version_need_no_gpu():
    L = corr.lib()
    assert L.mwax_corr_strerror(0) == b"ok"
    assert b"unsupported" in L.mwax_corr_strerror(-3)
    assert b"sm_100a" in L.mwax_corr_version()


def test_argument_validation_is_synchronous_and_needs_no_gpu():
    L = corr.lib()
    # invalid sizes and unsupported FFT lengths are rejected before any device is touched
    assert not L.mwax_corr_create(0, 64, 64, 1, 1) and L.mwax_corr_last_error() == -2
    assert not L.mwax_corr_create(16, 96, 96, 1, 1) and L.mwax_corr_last_error() == -3      # 96 = 2^5 * 3
    assert not L.mwax_corr_create(16, 12800, 64, 1, 1) and L.mwax_corr_last_error() == -3   # > 6400
    assert not L.mwax_corr_create(16, 64, 128, 1, 1) and L.mwax_corr_last_error() == -3     # keep > fft
    assert not L.mwax_corr_create(16, 64, 64, 1, 3) and L.mwax_corr_last_error() == -3      # 3 does not divide 64
    assert not L.mwax_xcorr_i8_create(12, 4, 70000) and L.mwax_corr_last_error() == -3      # int32 could overflow
    assert not L.mwax_xcorr_i8_create(0, 4, 100) and L.mwax_corr_last_error() == -2
    assert L.mwax_corr_destroy(None) == 0 and L.mwax_xcorr_i8_destroy(None) == 0
    assert L.mwax_corr_process(None, None, None, None) == -1


def test_static_entry_validates_sizes_without_a_gpu_and_calls_no_allocator():
    """mwax_corr_process_static: the size limit is checked before any device is touched, and the function's source has no
    allocating call (the scratch is a static device array whose address comes from cudaGetSymbolAddress)."""
    import ctypes
    L = corr.lib()
    buf = ctypes.create_string_buffer(64)
    a = (ctypes.addressof(buf) + 15) & ~15
    assert L.mwax_corr_static_workspace_max() == 32 * 1024 * 1024
    assert L.mwax_corr_process_static(a, a, 128, 128, 513, 1, None) == -7            # 128 x 513 x 256 x 2 B > 32 MiB
    assert b"static workspace" in L.mwax_corr_strerror(-7)
    assert L.mwax_corr_process_static(a, a, 128, 100, 4, 1, None) == -3              # no register kernel for N = 100
    assert L.mwax_corr_process_static(a + 1, a, 128, 128, 4, 1, None) == -2          # misaligned voltages
    assert L.mwax_corr_process_static(None, a, 128, 128, 4, 1, None) == -1
    src = open(os.path.join(ROOT, "paper_2303_11557_b200", "csrc", "mwax_api.cu")).read()
    body = src[src.index("static __device__ __align__(256)"):]
    assert "cudaGetSymbolAddress" in body
    for banned in ("cudaMalloc", "cudaFree", "cudaMemcpy", "upload("):
        assert banned not in body, banned


def test_library_reads_no_environment_variables():
    """Every knob is an argument or a set_option key (include/mwax_corr.h): no getenv in the product sources."""
    csrc = os.path.join(ROOT, "paper_2303_11557_b200", "csrc")
    for f in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, f)).read(), f"{f} reads the environment"
    hdr = open(HEADER).read()
    for opt in ("MWAX_OPT_AVG_MODE", "MWAX_OPT_ACCUMULATE", "MWAX_OPT_DC_EXCLUDE", "MWAX_OPT_X_EDGE_RUNS"):
        assert opt in hdr and hasattr(corr, opt)


def test_product_path_fails_loudly_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(corr.MwaxError):
        corr.MwaxCorr(16, 64, 64, 4, 1)     # MWAX_ERR_ARCH: there is no CPU fallback


def test_product_does_not_import_the_oracle():
    """The product shares no code with the oracle and never routes through it."""
    pkg = os.path.join(ROOT, "paper_2303_11557_b200")
    pat = re.compile(r"(from\s+oracle|import\s+oracle|libmwax_oracle|mwax_oracle_|#include\s+[\"<].*oracle)")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".c", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not pat.search(text), f"{f} references the oracle"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2303_11557_b200" not in text and "from paper_2303_11557_b200" not in text

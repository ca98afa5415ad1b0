"""CPU tests of the C-ABI boundary: libfdas.so loads, exports every function include/fdas.h declares, the
Python binding names the same set, and argument validation / error reporting work without a GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1711_10855_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "fdas.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fdas_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = declared_functions()
    assert "fdas_plan_create" in names and "fdas_convolve" in names and "fdas_set_templates" in names
    assert "fdas_plan_destroy" in names and len(names) >= 15
    lib = ctypes.CDLL(B.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"{n} is declared in include/fdas.h but not exported by libfdas.so"
    assert sorted(B.SYMBOLS) == names, "binding.SYMBOLS and include/fdas.h disagree"


def test_status_strings_and_version():
    assert B.status_string(B.FDAS_OK) == "FDAS_OK"
    assert B.status_string(B.FDAS_ERR_NO_TEMPLATES) == "FDAS_ERR_NO_TEMPLATES"
    assert B.status_string(77) == "FDAS_ERR_UNKNOWN"
    assert "sm_100a" in B.version()


@pytest.mark.parametrize("args,status", [
    ((0, 4, 2, 64, 512), B.FDAS_ERR_INVALID_ARG),          # n_f < 1
    ((1000, -2, 2, 64, 512), B.FDAS_ERR_INVALID_ARG),      # z_max < 0
    ((1000, 4, 0, 64, 512), B.FDAS_ERR_INVALID_ARG),       # z_step < 1
    ((1000, 5, 2, 64, 512), B.FDAS_ERR_INVALID_ARG),       # z_max not a multiple of z_step
    ((1000, 4, 2, 63, 512), B.FDAS_ERR_INVALID_ARG),       # odd template width
    ((1000, 4, 2, 0, 512), B.FDAS_ERR_INVALID_ARG),        # width < 2
    ((1000, 4, 2, 300, 512), B.FDAS_ERR_INVALID_ARG),      # width > L/2
    ((1000, 4, 2, 64, 500), B.FDAS_ERR_INVALID_ARG),       # L not a power of two
    ((1000, 4, 2, 64, 256), B.FDAS_ERR_UNSUPPORTED),       # power of two but not offered
    ((1000, 4, 2, 64, 16384), B.FDAS_ERR_UNSUPPORTED),
])
def test_plan_create_validates_before_touching_the_gpu(args, status):
    out = ctypes.c_void_p()
    s = B.lib().fdas_plan_create(ctypes.byref(out), *args)
    assert s == status and not out.value
    assert B.lib().fdas_plan_create(None, 1000, 4, 2, 64, 512) == B.FDAS_ERR_INVALID_ARG


def test_null_plans_are_handled():
    L = B.lib()
    assert L.fdas_plan_destroy(None) == B.FDAS_OK
    assert L.fdas_plan_nz(None) == 0 and L.fdas_plan_step(None) == 0 and L.fdas_plan_nseg(None) == 0
    assert L.fdas_plan_set_batch(None, 2) == B.FDAS_ERR_INVALID_ARG
    assert L.fdas_set_templates(None, None) == B.FDAS_ERR_INVALID_ARG
    assert L.fdas_convolve(None, None, None, None) == B.FDAS_ERR_INVALID_ARG
    assert L.fdas_convolve_host(None, None, None, None) == B.FDAS_ERR_INVALID_ARG
    assert L.fdas_debug_fft(4096, 1, None, None, 0) == B.FDAS_ERR_INVALID_ARG
    assert L.fdas_debug_fft(300, 1, 8, 8, 0) == B.FDAS_ERR_UNSUPPORTED


def test_no_cpu_fallback_without_a_gpu():
    """On a box without a CUDA device a valid plan cannot be created: the library fails loudly
    (FDAS_ERR_CUDA / FDAS_ERR_ALLOC) instead of computing anything on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(B.FdasError) as e:
        B.Plan(1 << 12, 4, 2, 64, 512)
    assert e.value.status in (B.FDAS_ERR_CUDA, B.FDAS_ERR_ALLOC)


def test_round2_entries_validate_before_touching_the_gpu():
    """The entry points added in round 2: NULL handling and argument checks that need no device."""
    L = B.lib()
    assert L.fdas_convolve_complex(None, None, None, None) == B.FDAS_ERR_INVALID_ARG
    assert L.fdas_detect_blockmax(None, None, None, None, None) == B.FDAS_ERR_INVALID_ARG
    assert L.fdas_detect_blockmax_host(None, None, None, None, None) == B.FDAS_ERR_INVALID_ARG
    assert L.fdas_plan_set_symmetry(None, 1) == B.FDAS_ERR_INVALID_ARG
    assert L.fdas_detect_candidates(None, None, 1.0, 8, None, None, None) == B.FDAS_ERR_INVALID_ARG
    assert L.fdas_detect_candidates_host(None, None, 1.0, 8, None, None, None) == B.FDAS_ERR_INVALID_ARG
    assert B.CANDIDATE_DTYPE.itemsize == 16
    assert L.fdas_plan_symmetry_active(None) == 0 and L.fdas_plan_grid(None) == 0
    out = ctypes.c_void_p()
    # stand-alone FFT: (n, elements per thread) combinations that do not exist
    for n, e, status in [(1000, 0, B.FDAS_ERR_UNSUPPORTED), (256, 0, B.FDAS_ERR_UNSUPPORTED), (4096, 8, B.FDAS_ERR_UNSUPPORTED),
                         (512, 16, B.FDAS_ERR_UNSUPPORTED), (1024, 4, B.FDAS_ERR_UNSUPPORTED)]:
        assert L.fdas_fft_plan_create(ctypes.byref(out), n, e) == status and not out.value
    assert L.fdas_fft_plan_create(None, 1024, 0) == B.FDAS_ERR_INVALID_ARG
    assert L.fdas_fft_exec(None, 1, 8, 16, 0, None) == B.FDAS_ERR_INVALID_ARG
    assert L.fdas_fft_plan_destroy(None) == B.FDAS_OK and L.fdas_fft_plan_grid(None) == 0
    # spectrum step: sample counts that are not powers of two, or outside 2^19 .. 2^27
    for n, status in [(0, B.FDAS_ERR_INVALID_ARG), (3 << 20, B.FDAS_ERR_INVALID_ARG), (1 << 18, B.FDAS_ERR_UNSUPPORTED),
                      (1 << 28, B.FDAS_ERR_UNSUPPORTED)]:
        assert L.fdas_spectrum_plan_create(ctypes.byref(out), n, 4096) == status and not out.value
    assert L.fdas_spectrum_exec(None, None, None, None) == B.FDAS_ERR_INVALID_ARG
    assert L.fdas_spectrum_plan_destroy(None) == B.FDAS_OK and L.fdas_spectrum_plan_bins(None) == 0
    assert L.fdas_debug_alu_peak(0, None, None) == B.FDAS_ERR_INVALID_ARG

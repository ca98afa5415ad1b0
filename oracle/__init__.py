"""FDAS oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes + numpy wrappers around oracle/fdas_oracle.c, the plain double-precision CPU statement of
eq.(2) of arXiv:1711.10855 (direct summation), its templates, and a double overlap-and-save.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import
this package.  It imports nothing from paper_1711_10855_b200 and that package imports nothing from
here.  Every wrapper only marshals arrays; the arithmetic is in the C file, which cites the passage
each function follows.
"""
import ctypes
import os

import numpy as np

from . import build as _build

_LIB = None


def lib():
    global _LIB
    if _LIB is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        dp = ctypes.POINTER(ctypes.c_double)
        i64 = ctypes.c_int64
        L.fdas_oracle_num_threads.restype = ctypes.c_int
        L.fdas_oracle_dft.argtypes = [dp, i64, ctypes.c_int, dp]
        L.fdas_oracle_dft.restype = None
        L.fdas_oracle_fft.argtypes = [dp, i64, ctypes.c_int]
        L.fdas_oracle_fft.restype = ctypes.c_int
        L.fdas_oracle_fresnel.argtypes = [ctypes.c_double, dp, dp]
        L.fdas_oracle_fresnel.restype = None
        L.fdas_oracle_response.argtypes = [ctypes.c_double, ctypes.c_double, dp, dp]
        L.fdas_oracle_response.restype = None
        L.fdas_oracle_templates.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp]
        L.fdas_oracle_templates.restype = ctypes.c_int
        L.fdas_oracle_direct.argtypes = [dp, i64, dp, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                         i64, i64, dp, dp]
        L.fdas_oracle_direct.restype = ctypes.c_int
        L.fdas_oracle_ols.argtypes = [dp, i64, dp, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                      ctypes.c_int, ctypes.c_int, dp]
        L.fdas_oracle_spectrum.argtypes = [dp, i64, i64, dp]
        L.fdas_oracle_spectrum.restype = ctypes.c_int
        L.fdas_oracle_blockmax.argtypes = [dp, ctypes.c_int, i64, i64, ctypes.c_int, dp, ctypes.POINTER(ctypes.c_int64)]
        L.fdas_oracle_blockmax.restype = ctypes.c_int
        L.fdas_oracle_ols.restype = ctypes.c_int
        _LIB = L
    return _LIB


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _c128(a):
    """complex array -> contiguous complex128 (viewed by C as interleaved doubles)."""
    return np.ascontiguousarray(np.asarray(a), dtype=np.complex128)


def num_threads() -> int:
    return int(lib().fdas_oracle_num_threads())


def dft(x, sign=-1):
    """eq.(3) by brute force; sign=+1 is the unnormalised inverse."""
    x = _c128(x)
    out = np.empty_like(x)
    lib().fdas_oracle_dft(_dp(x), x.size, int(sign), _dp(out))
    return out


def fft(x, sign=-1):
    """eq.(3) by recursive radix-2 (length must be a power of two)."""
    x = _c128(x).copy()
    if lib().fdas_oracle_fft(_dp(x), x.size, int(sign)) != 0:
        raise ValueError("oracle fft: length must be a power of two")
    return x


def fresnel(x):
    """(C(x), S(x)), the pi t^2/2 convention."""
    c = ctypes.c_double()
    s = ctypes.c_double()
    lib().fdas_oracle_fresnel(float(x), ctypes.byref(c), ctypes.byref(s))
    return c.value, s.value


def response(q, z):
    """I(q,z) = int_0^1 exp(i pi (2 q u + z u^2)) du."""
    re = ctypes.c_double()
    im = ctypes.c_double()
    lib().fdas_oracle_response(float(q), float(z), ctypes.byref(re), ctypes.byref(im))
    return complex(re.value, im.value)


def templates(z_max, z_step, m):
    """Unit-normalised template bank, complex128 [n_z][m]; row i <-> z = -z_max + i*z_step."""
    if z_step < 1 or z_max < 0 or z_max % z_step:
        raise ValueError("bad z grid")
    n_z = 2 * z_max // z_step + 1
    out = np.empty((n_z, m), dtype=np.complex128)
    if lib().fdas_oracle_templates(int(z_max), int(z_step), int(m), _dp(out)) != n_z:
        raise ValueError("oracle templates: bad arguments")
    return out


def direct(spectrum, templates_, rows=None, cols=None, want="power"):
    """eq.(2) by direct summation on rows [r0,r1) x columns [c0,c1) of the plane.

    spectrum: complex [n_f]; templates_: complex [n_z][m].  Returns float64 power [rows][cols]
    (want="power"), complex128 amplitude A' (want="amp"), or both as a tuple (want="both").
    """
    A = _c128(spectrum)
    H = _c128(templates_)
    n_z, m = H.shape
    r0, r1 = (0, n_z) if rows is None else rows
    c0, c1 = (0, A.size) if cols is None else cols
    nr, nc = r1 - r0, c1 - c0
    p = np.empty((nr, nc), dtype=np.float64) if want in ("power", "both") else None
    a = np.empty((nr, nc), dtype=np.complex128) if want in ("amp", "both") else None
    rc = lib().fdas_oracle_direct(_dp(A), A.size, _dp(H), m, r0, nr, c0, nc,
                                  _dp(p) if p is not None else None,
                                  _dp(a) if a is not None else None)
    if rc != 0:
        raise ValueError("oracle direct: bad arguments")
    if want == "power":
        return p
    if want == "amp":
        return a
    return p, a


def ols(spectrum, templates_, seg_len, step=None, rows=None):
    """The same plane by double-precision overlap-and-save; float64 [rows][n_f]."""
    A = _c128(spectrum)
    H = _c128(templates_)
    n_z, m = H.shape
    if step is None:
        step = seg_len - m + 1
    r0, r1 = (0, n_z) if rows is None else rows
    p = np.empty((r1 - r0, A.size), dtype=np.float64)
    rc = lib().fdas_oracle_ols(_dp(A), A.size, _dp(H), m, r0, r1 - r0, int(seg_len), int(step), _dp(p))
    if rc != 0:
        raise ValueError("oracle ols: bad arguments")
    return p


def blockmax(power, blk, float32_decision=True):
    """Detection step over a power plane [rows][cols] (reading 17): per row and block of `blk`
    columns the maximum and the lowest in-block offset attaining it.  Returns (float64 [rows][n_blk],
    int64 [rows][n_blk]).  float32_decision: compare float32-rounded powers (the CUDA path's precision)."""
    p = np.ascontiguousarray(power, dtype=np.float64)
    if p.ndim != 2:
        raise ValueError("power must be [rows][cols]")
    n_rows, n_cols = p.shape
    if int(blk) < 1 or n_cols < 1:
        raise ValueError("oracle blockmax: bad arguments")
    n_blk = (n_cols + int(blk) - 1) // int(blk)
    mx = np.empty((n_rows, n_blk), dtype=np.float64)
    ar = np.empty((n_rows, n_blk), dtype=np.int64)
    rc = lib().fdas_oracle_blockmax(_dp(p), n_rows, n_cols, int(blk), int(bool(float32_decision)), _dp(mx),
                                    ar.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)))
    if rc != 0:
        raise ValueError("oracle blockmax: bad arguments")
    return mx, ar


def candidates(power, blk, threshold, capacity):
    """Thresholded candidate list over a power plane [rows][cols] (reading 20; "detect"):
    every block maximum of reading 17 whose float32 power is >= float32(threshold) is a candidate
    (row, column = block * blk + offset, power as the float32 value the plane holds).  The list is ordered by (row, column); the first `capacity`
    entries are kept.  Returns (n_found, rows int64 [n_kept], cols int64 [n_kept], powers float64 [n_kept]);
    n_found counts every candidate, kept or not (n_found - n_kept is the overflow).
    Written out step by step on top of blockmax: threshold, order, truncate."""
    mx, ar = blockmax(power, blk, float32_decision=True)
    thr = np.float32(threshold)
    found = []
    for r in range(mx.shape[0]):            # rows in order, blocks in order: (row, column) ascending
        for b in range(mx.shape[1]):
            if np.float32(mx[r, b]) >= thr:
                found.append((r, b * int(blk) + int(ar[r, b]), float(mx[r, b])))
    kept = found[:max(0, int(capacity))]
    return (len(found), np.array([k[0] for k in kept], dtype=np.int64), np.array([k[1] for k in kept], dtype=np.int64),
            np.array([k[2] for k in kept], dtype=np.float64))


def spectrum(series, whiten_block=0):
    """P:21 "the FFT output of the observation" (reading 18): eq.(3) of the real series, bins
    0 .. n_t/2 - 1, whitened in blocks of `whiten_block` bins (0: not whitened).  complex128 [n_t/2]."""
    x = np.ascontiguousarray(series, dtype=np.float64)
    if x.ndim != 1:
        raise ValueError("series must be one-dimensional")
    out = np.empty(x.size // 2, dtype=np.complex128)
    rc = lib().fdas_oracle_spectrum(_dp(x), x.size, int(whiten_block), _dp(out))
    if rc != 0:
        raise ValueError("oracle spectrum: bad arguments")
    return out

"""Thin ctypes binding over libfdas.so (include/fdas.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used by callers for device
memory and streams; this module only needs `.data_ptr()` / `.cuda_stream` from them.  If libfdas.so
is missing this module raises on first use -- there is no fallback.
"""
import ctypes
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libfdas.so")

FDAS_OK, FDAS_ERR_INVALID_ARG, FDAS_ERR_UNSUPPORTED, FDAS_ERR_ALLOC, FDAS_ERR_NO_TEMPLATES, FDAS_ERR_CUDA = range(6)
FDAS_ERR_TOO_LARGE = 6
NOALLOC_MAX_BANK = 1 << 20  # FDAS_NOALLOC_MAX_BANK: n_z * segment_len that fdas_convolve_noalloc accepts

# every symbol include/fdas.h declares: name -> (restype, argtypes)
_vp, _i64, _int = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
SYMBOLS = {
    "fdas_plan_create": (_int, [ctypes.POINTER(_vp), _i64, _int, _int, _int, _int]),
    "fdas_plan_set_batch": (_int, [_vp, _int]),
    "fdas_set_templates": (_int, [_vp, _vp]),
    "fdas_plan_set_symmetry": (_int, [_vp, _int]),
    "fdas_plan_symmetry_active": (_int, [_vp]),
    "fdas_convolve": (_int, [_vp, _vp, _vp, _vp]),
    "fdas_convolve_noalloc": (_int, [_i64, _int, _int, _int, _int, _int, _vp, _vp, _vp, _vp]),
    "fdas_convolve_host": (_int, [_vp, _vp, _vp, _vp]),
    "fdas_convolve_complex": (_int, [_vp, _vp, _vp, _vp]),
    "fdas_detect_blockmax": (_int, [_vp, _vp, _vp, _vp, _vp]),
    "fdas_detect_blockmax_host": (_int, [_vp, _vp, _vp, _vp, _vp]),
    "fdas_detect_candidates": (_int, [_vp, _vp, ctypes.c_float, _int, _vp, _vp, _vp]),
    "fdas_detect_candidates_host": (_int, [_vp, _vp, ctypes.c_float, _int, _vp, _vp, _vp]),
    "fdas_plan_destroy": (_int, [_vp]),
    "fdas_plan_nz": (_int, [_vp]),
    "fdas_plan_step": (_int, [_vp]),
    "fdas_plan_nseg": (_i64, [_vp]),
    "fdas_plan_batch": (_int, [_vp]),
    "fdas_plan_grid": (_int, [_vp]),
    "fdas_plan_last_launch_count": (_int, [_vp]),
    "fdas_plan_last_cuda_error": (_int, [_vp]),
    "fdas_status_string": (ctypes.c_char_p, [_int]),
    "fdas_fft_plan_create": (_int, [ctypes.POINTER(_vp), _int, _int]),
    "fdas_fft_exec": (_int, [_vp, _i64, _vp, _vp, _int, _vp]),
    "fdas_fft_exec_many": (_int, [_vp, _int, _i64, _vp, _vp, _int, _vp]),
    "fdas_fft_plan_destroy": (_int, [_vp]),
    "fdas_fft_plan_elems_per_thread": (_int, [_vp]),
    "fdas_fft_plan_grid": (_int, [_vp]),
    "fdas_spectrum_plan_create": (_int, [ctypes.POINTER(_vp), _i64, _i64]),
    "fdas_spectrum_exec": (_int, [_vp, _vp, _vp, _vp]),
    "fdas_spectrum_plan_destroy": (_int, [_vp]),
    "fdas_spectrum_plan_bins": (_i64, [_vp]),
    "fdas_debug_fft": (_int, [_int, _i64, _vp, _vp, _int]),
    "fdas_debug_layout": (_i64, [_int, _int, _int, _int, _int]),
    "fdas_debug_alu_peak": (_int, [_int, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]),
    "fdas_version": (ctypes.c_char_p, []),
}

# fdas_candidate (include/fdas.h): view a uint8 / int32 buffer of 16-byte records with this dtype
CANDIDATE_DTYPE = np.dtype([("item", np.int32), ("row", np.int32), ("column", np.int32), ("power", np.float32)])

_LIB = None


class FdasError(RuntimeError):
    def __init__(self, status, where):
        self.status = int(status)
        super().__init__(f"{where}: {status_string(status)}")


def lib():
    """Load libfdas.so (never builds it; see paper_1711_10855_b200.build)."""
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1711_10855_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _LIB = L
    return _LIB


def status_string(s) -> str:
    return lib().fdas_status_string(int(s)).decode()


def version() -> str:
    return lib().fdas_version().decode()


def _check(s, where):
    if s != FDAS_OK:
        raise FdasError(s, where)


def _ptr(x):
    """Device/host address of a torch tensor, numpy array, int or None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    raise TypeError(type(x))


def _stream(s):
    if s is None:
        return None
    if isinstance(s, int):
        return s
    return s.cuda_stream  # torch.cuda.Stream


class Plan:
    """fdas_plan_create ... fdas_plan_destroy as a Python object (same names, same arguments)."""

    def __init__(self, n_f, z_max, z_step, template_width, segment_len, n_batch=1):
        self._h = _vp()
        _check(lib().fdas_plan_create(ctypes.byref(self._h), int(n_f), int(z_max), int(z_step),
                                      int(template_width), int(segment_len)), "fdas_plan_create")
        self.n_f, self.m, self.L = int(n_f), int(template_width), int(segment_len)
        if n_batch != 1:
            self.set_batch(n_batch)

    # geometry
    @property
    def n_z(self): return lib().fdas_plan_nz(self._h)
    @property
    def step(self): return lib().fdas_plan_step(self._h)
    @property
    def n_seg(self): return lib().fdas_plan_nseg(self._h)
    @property
    def n_batch(self): return lib().fdas_plan_batch(self._h)
    @property
    def grid(self): return lib().fdas_plan_grid(self._h)
    @property
    def last_launch_count(self): return lib().fdas_plan_last_launch_count(self._h)
    @property
    def last_cuda_error(self): return lib().fdas_plan_last_cuda_error(self._h)

    def set_batch(self, n_batch):
        _check(lib().fdas_plan_set_batch(self._h, int(n_batch)), "fdas_plan_set_batch")

    def set_symmetry(self, enable):
        _check(lib().fdas_plan_set_symmetry(self._h, int(bool(enable))), "fdas_plan_set_symmetry")

    @property
    def symmetry_active(self): return bool(lib().fdas_plan_symmetry_active(self._h))

    def set_templates(self, h_templates):
        """h_templates: complex64 [n_z][m] numpy array (HOST)."""
        h = np.ascontiguousarray(h_templates, dtype=np.complex64)
        if h.shape != (self.n_z, self.m):
            raise ValueError(f"templates must be [{self.n_z}][{self.m}], got {h.shape}")
        _check(lib().fdas_set_templates(self._h, h.ctypes.data), "fdas_set_templates")

    def convolve(self, d_spectrum, d_power, stream=None):
        """d_spectrum: DEVICE complex64 [n_batch][n_f]; d_power: DEVICE float32 [n_batch][n_z][n_f]."""
        _check(lib().fdas_convolve(self._h, _ptr(d_spectrum), _ptr(d_power), _stream(stream)), "fdas_convolve")

    def convolve_host(self, h_spectrum, h_power, stream=None):
        """HOST buffers (pinned torch tensors or numpy arrays); copies are inside the call."""
        _check(lib().fdas_convolve_host(self._h, _ptr(h_spectrum), _ptr(h_power), _stream(stream)),
               "fdas_convolve_host")

    def convolve_complex(self, d_spectrum, d_amp, stream=None):
        """d_amp: DEVICE complex64 [n_batch][n_z][n_f], the filtered spectrum A' of eq.(2)."""
        _check(lib().fdas_convolve_complex(self._h, _ptr(d_spectrum), _ptr(d_amp), _stream(stream)), "fdas_convolve_complex")

    def detect_blockmax(self, d_spectrum, d_max, d_arg, stream=None):
        """d_max float32, d_arg int32: DEVICE [n_batch][n_z][n_seg]; blocks of `step` columns."""
        _check(lib().fdas_detect_blockmax(self._h, _ptr(d_spectrum), _ptr(d_max), _ptr(d_arg), _stream(stream)),
               "fdas_detect_blockmax")

    def detect_blockmax_host(self, h_spectrum, h_max, h_arg, stream=None):
        _check(lib().fdas_detect_blockmax_host(self._h, _ptr(h_spectrum), _ptr(h_max), _ptr(h_arg), _stream(stream)),
               "fdas_detect_blockmax_host")

    def detect_candidates(self, d_spectrum, threshold, capacity, d_cand, d_count, stream=None):
        """d_cand: DEVICE [capacity] records of CANDIDATE_DTYPE (16 bytes); d_count: DEVICE int32 [2] = (found, written)."""
        _check(lib().fdas_detect_candidates(self._h, _ptr(d_spectrum), float(threshold), int(capacity), _ptr(d_cand), _ptr(d_count),
                                            _stream(stream)), "fdas_detect_candidates")

    def detect_candidates_host(self, h_spectrum, threshold, capacity, h_cand, h_count, stream=None):
        _check(lib().fdas_detect_candidates_host(self._h, _ptr(h_spectrum), float(threshold), int(capacity), _ptr(h_cand),
                                                 _ptr(h_count), _stream(stream)), "fdas_detect_candidates_host")

    def destroy(self):
        if self._h:
            lib().fdas_plan_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class FftPlan:
    """fdas_fft_plan_create ... fdas_fft_plan_destroy: the stand-alone batched segment FFT."""

    def __init__(self, n, elems_per_thread=0):
        self._h = _vp()
        _check(lib().fdas_fft_plan_create(ctypes.byref(self._h), int(n), int(elems_per_thread)), "fdas_fft_plan_create")
        self.n = int(n)

    @property
    def elems_per_thread(self): return lib().fdas_fft_plan_elems_per_thread(self._h)
    @property
    def grid(self): return lib().fdas_fft_plan_grid(self._h)

    def exec(self, n_fft, d_in, d_out, inverse=False, stream=None):
        _check(lib().fdas_fft_exec(self._h, int(n_fft), _ptr(d_in), _ptr(d_out), int(bool(inverse)), _stream(stream)),
               "fdas_fft_exec")

    def exec_many(self, n_launches, n_fft, d_in, d_out, inverse=False, stream=None):
        _check(lib().fdas_fft_exec_many(self._h, int(n_launches), int(n_fft), _ptr(d_in), _ptr(d_out), int(bool(inverse)),
                                        _stream(stream)), "fdas_fft_exec_many")

    def destroy(self):
        if self._h:
            lib().fdas_fft_plan_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class SpectrumPlan:
    """fdas_spectrum_plan_create ... _destroy: real time series -> whitened complex spectrum."""

    def __init__(self, n_samples, whiten_block=0):
        self._h = _vp()
        _check(lib().fdas_spectrum_plan_create(ctypes.byref(self._h), int(n_samples), int(whiten_block)),
               "fdas_spectrum_plan_create")

    @property
    def bins(self): return lib().fdas_spectrum_plan_bins(self._h)

    def exec(self, d_series, d_spectrum, stream=None):
        _check(lib().fdas_spectrum_exec(self._h, _ptr(d_series), _ptr(d_spectrum), _stream(stream)), "fdas_spectrum_exec")

    def destroy(self):
        if self._h:
            lib().fdas_spectrum_plan_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def convolve_noalloc(n_f, n_batch, z_max, z_step, template_width, segment_len, d_templates, d_spectrum, d_power, stream=None):
    """fdas_convolve_noalloc: plan-less fdas_convolve that allocates nothing (scratch inside libfdas.so).

    For hosts that cannot call cudaMalloc while they run (all device memory handed out at start-up, or owned by a
    framework's pool).  d_templates: DEVICE complex64 [n_z][m]; the other buffers as Plan.convolve.  Raises
    FdasError(FDAS_ERR_TOO_LARGE) when n_z * segment_len > NOALLOC_MAX_BANK.  Calls on one GPU share one scratch
    array: keep them on one stream.  Make the first call on a GPU outside any stream capture.
    """
    _check(lib().fdas_convolve_noalloc(int(n_f), int(n_batch), int(z_max), int(z_step), int(template_width), int(segment_len),
                                       _ptr(d_templates), _ptr(d_spectrum), _ptr(d_power), _stream(stream)),
           "fdas_convolve_noalloc")


def debug_fft(segment_len, n_seg, d_in, d_out, inverse=False):
    _check(lib().fdas_debug_fft(int(segment_len), int(n_seg), _ptr(d_in), _ptr(d_out), int(bool(inverse))),
           "fdas_debug_fft")


# `what` selectors of fdas_debug_layout (include/fdas.h)
(LAYOUT_GEOMETRY, LAYOUT_FREQ, LAYOUT_GMOD, LAYOUT_TWA, LAYOUT_FIX, LAYOUT_SHFL_SRC, LAYOUT_SHFL_DST,
 LAYOUT_WRITE_A, LAYOUT_READ_A, LAYOUT_WRITE_B, LAYOUT_READ_B, LAYOUT_TW_MID) = range(12)


def debug_layout(segment_len, what, t=0, a=0, b=0) -> int:
    """Host evaluation of the kernels' index maps (no GPU needed); -1 = out of range."""
    return int(lib().fdas_debug_layout(int(segment_len), int(what), int(t), int(a), int(b)))


def debug_alu_peak(packed=False):
    """(TFLOP/s, ms) of the register-only FMA chains of fdas_debug_alu_peak."""
    tf, ms = ctypes.c_double(), ctypes.c_double()
    _check(lib().fdas_debug_alu_peak(int(bool(packed)), ctypes.byref(tf), ctypes.byref(ms)), "fdas_debug_alu_peak")
    return tf.value, ms.value

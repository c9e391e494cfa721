"""Thin ctypes binding over the C ABI of include/fdd.h -- argument marshalling only.

Every step of the hot path runs in the CUDA library (``csrc/libfdd_b200.so``); PyTorch is used
by callers only to own device memory and streams.  There is no CPU fallback: if the library is
missing or no CUDA device is present, creating a plan raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence, Tuple

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "csrc", "libfdd_b200.so")

FDD_MODE_TIME, FDD_MODE_FOURIER = 0, 1
FDD_KERNEL_AUTO, FDD_KERNEL_GENERIC, FDD_KERNEL_SYMMETRIC, FDD_KERNEL_SYMMETRIC2 = 0, 1, 2, 3
FDD_KERNEL_MIXED = 4
FDD_KERNEL_TENSOR = 5
FDD_INVERSE_CUFFT, FDD_INVERSE_TWO_PASS, FDD_INVERSE_AUTO = 0, 1, 2
FDD_OK = 0
FDD_ERR_TOO_LARGE = -6
FDD_STATIC_MAX_PHASES = 1 << 20
FDD_NUM_STAGES = 6
STAGE_NAMES = ("unpack", "r2c", "rotate_sum", "c2r", "tdd_transpose", "tdd_shift_add")

EXPORTS = (
    "fdd_plan_create", "fdd_plan_create_from_delays", "fdd_plan_set_kdm", "fdd_plan_set_kernel",
    "fdd_plan_set_decimation", "fdd_plan_get_output_shape", "fdd_plan_prepare",
    "fdd_plan_set_y_budget", "fdd_plan_set_inverse", "fdd_plan_get_inverse",
    "fdd_execute", "fdd_execute_host", "fdd_execute_beams", "fdd_tdd_execute", "fdd_plan_destroy", "fdd_plan_get_info",
    "fdd_plan_get_delays", "fdd_plan_set_profiling", "fdd_plan_get_stage_ms",
    "fdd_plan_get_spectrum", "fdd_plan_get_padding", "fdd_rotate_sum_only", "fdd_measure_fp32_peak", "fdd_tc_selftest",
    "fdd_rotate_sum_static", "fdd_error_string",
)


class FddError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {error_string(status)} (status {status})")


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen the C-ABI library and declare its prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(
            f"{LIB_PATH} not built: run `python -m paper_2110_03482_b200.build` "
            "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    c_int, c_ll, c_dbl, vp = ctypes.c_int, ctypes.c_longlong, ctypes.c_double, ctypes.c_void_p
    P = ctypes.POINTER
    lib.fdd_plan_create.argtypes = [P(vp), c_int, c_ll, c_dbl, c_dbl, c_dbl, P(c_dbl), c_int]
    lib.fdd_plan_create_from_delays.argtypes = [P(vp), c_int, c_ll, P(c_dbl), c_int]
    lib.fdd_plan_set_kdm.argtypes = [vp, c_dbl]
    lib.fdd_plan_set_kernel.argtypes = [vp, c_int]
    lib.fdd_execute.argtypes = [vp, vp, vp, c_int, vp]
    lib.fdd_execute_host.argtypes = [vp, vp, vp, c_int, vp]
    lib.fdd_execute_beams.argtypes = [vp, vp, vp, c_int, c_int, vp]
    lib.fdd_tdd_execute.argtypes = [vp, vp, vp, vp]
    lib.fdd_plan_destroy.argtypes = [vp]
    lib.fdd_plan_get_info.argtypes = [vp, P(c_ll), P(c_ll), P(c_ll), P(c_dbl),
                                      P(ctypes.c_size_t), P(c_int)]
    lib.fdd_plan_get_delays.argtypes = [vp, P(c_dbl)]
    lib.fdd_plan_set_profiling.argtypes = [vp, c_int]
    lib.fdd_plan_set_decimation.argtypes = [vp, c_int]
    lib.fdd_plan_prepare.argtypes = [vp, c_int]
    lib.fdd_plan_set_y_budget.argtypes = [vp, ctypes.c_size_t]
    lib.fdd_plan_set_inverse.argtypes = [vp, c_int]
    lib.fdd_plan_get_inverse.argtypes = [vp, P(c_int)]
    lib.fdd_plan_get_output_shape.argtypes = [vp, ctypes.POINTER(ctypes.c_longlong),
                                              ctypes.POINTER(ctypes.c_longlong)]
    lib.fdd_plan_get_stage_ms.argtypes = [vp, P(ctypes.c_float), P(c_int)]
    lib.fdd_plan_get_spectrum.argtypes = [vp, P(vp), P(c_ll), P(c_dbl)]
    lib.fdd_rotate_sum_only.argtypes = [vp, vp, c_int, vp]
    lib.fdd_plan_get_padding.argtypes = [vp, P(c_ll)]
    lib.fdd_tc_selftest.argtypes = [vp, vp, vp, vp]
    lib.fdd_rotate_sum_static.argtypes = [vp, c_ll, vp, c_int, c_ll, c_ll, c_int, vp, ctypes.c_float, vp]
    lib.fdd_measure_fp32_peak.argtypes = [c_int, c_int, P(c_dbl), P(ctypes.c_float)]
    for name in EXPORTS:
        getattr(lib, name).restype = c_int
    lib.fdd_error_string.argtypes = [c_int]
    lib.fdd_error_string.restype = ctypes.c_char_p
    _lib = lib
    return lib


def error_string(status: int) -> str:
    return load_library().fdd_error_string(int(status)).decode()


def _check(status: int, where: str) -> None:
    if status != FDD_OK:
        raise FddError(status, where)


def _dbl_array(values) -> ctypes.Array:
    vals = [float(v) for v in values]
    return (ctypes.c_double * len(vals))(*vals)


def _ptr(t) -> int:
    """Device (or host) address of a torch tensor / numpy array / int."""
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def _stream_handle(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


class Plan:
    """Owner of one ``fdd_plan*``.  Methods carry the C ABI's names without the prefix."""

    def __init__(self, handle: int, nchans: int, nsamps: int, ndm: int):
        self._h = ctypes.c_void_p(handle)
        self.nchans, self.nsamps, self.ndm = nchans, nsamps, ndm
        nfft, nbins, valid, maxd, scratch, kernel = self.get_info()
        self.nfft, self.nbins = nfft, nbins

    # -- creation ------------------------------------------------------------------------
    @classmethod
    def create(cls, nchans: int, nsamps: int, tsamp: float, f_lo: float, f_hi: float,
               dm_list: Sequence[float]) -> "Plan":
        lib = load_library()
        h = ctypes.c_void_p()
        dms = _dbl_array(dm_list)
        _check(lib.fdd_plan_create(ctypes.byref(h), int(nchans), int(nsamps), float(tsamp),
                                   float(f_lo), float(f_hi), dms, len(dms)), "fdd_plan_create")
        return cls(h.value, int(nchans), int(nsamps), len(dms))

    @classmethod
    def create_from_delays(cls, nchans: int, nsamps: int, delays) -> "Plan":
        """``delays``: [ndm][nchans] samples (numpy array or nested sequence, host)."""
        import numpy as np
        lib = load_library()
        d = np.ascontiguousarray(delays, dtype=np.float64)
        if d.ndim != 2 or d.shape[1] != nchans:
            raise ValueError("delays must be [ndm][nchans]")
        h = ctypes.c_void_p()
        _check(lib.fdd_plan_create_from_delays(
            ctypes.byref(h), int(nchans), int(nsamps),
            d.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), d.shape[0]),
            "fdd_plan_create_from_delays")
        return cls(h.value, int(nchans), int(nsamps), d.shape[0])

    # -- C ABI, one method per entry point ---------------------------------------------------
    def set_kdm(self, k_dm: float) -> None:
        _check(load_library().fdd_plan_set_kdm(self._h, float(k_dm)), "fdd_plan_set_kdm")

    def set_kernel(self, kernel: int) -> None:
        _check(load_library().fdd_plan_set_kernel(self._h, int(kernel)), "fdd_plan_set_kernel")

    def execute(self, in_u8, out, mode: int = FDD_MODE_TIME, stream=None) -> None:
        """Device tensors in/out (see include/fdd.h for layouts); asynchronous on ``stream``."""
        _check(load_library().fdd_execute(self._h, _ptr(in_u8), _ptr(out), int(mode),
                                          _stream_handle(stream)), "fdd_execute")

    def execute_host(self, in_host, out_host, mode: int = FDD_MODE_TIME, stream=None) -> None:
        """Host buffers in/out; returns when the result has landed in ``out_host``."""
        _check(load_library().fdd_execute_host(self._h, _ptr(in_host), _ptr(out_host), int(mode),
                                               _stream_handle(stream)), "fdd_execute_host")

    def execute_beams(self, in_u8, out, nbeams: int, mode: int = FDD_MODE_TIME, stream=None) -> None:
        """Device tensors: in_u8 [nbeams][nsamps][nchans], out [nbeams][...]."""
        _check(load_library().fdd_execute_beams(self._h, _ptr(in_u8), _ptr(out), int(nbeams), int(mode),
                                                _stream_handle(stream)), "fdd_execute_beams")

    def tdd_execute(self, in_u8, out, stream=None) -> None:
        """The time-domain comparator (Eq. 2): device tensors, out float32 [ndm][nsamps]."""
        _check(load_library().fdd_tdd_execute(self._h, _ptr(in_u8), _ptr(out),
                                              _stream_handle(stream)), "fdd_tdd_execute")

    def rotate_sum_only(self, out, mode: int = FDD_MODE_FOURIER, stream=None) -> None:
        _check(load_library().fdd_rotate_sum_only(self._h, _ptr(out), int(mode),
                                                  _stream_handle(stream)), "fdd_rotate_sum_only")

    def get_info(self) -> Tuple[int, int, int, float, int, int]:
        """(nfft, nbins, valid_len, max_delay_samples, scratch_bytes, kernel)."""
        nfft, nbins, valid = ctypes.c_longlong(), ctypes.c_longlong(), ctypes.c_longlong()
        maxd, scratch, kernel = ctypes.c_double(), ctypes.c_size_t(), ctypes.c_int()
        _check(load_library().fdd_plan_get_info(
            self._h, ctypes.byref(nfft), ctypes.byref(nbins), ctypes.byref(valid),
            ctypes.byref(maxd), ctypes.byref(scratch), ctypes.byref(kernel)), "fdd_plan_get_info")
        return nfft.value, nbins.value, valid.value, maxd.value, scratch.value, kernel.value

    def get_delays(self):
        import numpy as np
        d = np.empty((self.ndm, self.nchans), dtype=np.float64)
        _check(load_library().fdd_plan_get_delays(
            self._h, d.ctypes.data_as(ctypes.POINTER(ctypes.c_double))), "fdd_plan_get_delays")
        return d

    def set_decimation(self, log2_factor: int) -> None:
        """Reduced-length inverse transform = down-sampling by 2^log2_factor."""
        _check(load_library().fdd_plan_set_decimation(self._h, int(log2_factor)),
               "fdd_plan_set_decimation")

    def prepare(self, mode: int = FDD_MODE_TIME) -> None:
        """Do every lazy allocation / upload of ``mode`` now, so execute never synchronises."""
        _check(load_library().fdd_plan_prepare(self._h, int(mode)), "fdd_plan_prepare")

    def set_inverse(self, which: int) -> None:
        """FDD_INVERSE_AUTO (default), FDD_INVERSE_CUFFT or FDD_INVERSE_TWO_PASS (hand-written, keeps the mean out of fp32)."""
        _check(load_library().fdd_plan_set_inverse(self._h, int(which)), "fdd_plan_set_inverse")

    def set_y_budget(self, nbytes: int) -> None:
        """Cap the TIME-mode Y scratch (trial DMs are then processed in chunks); 0 = default."""
        _check(load_library().fdd_plan_set_y_budget(self._h, int(nbytes)), "fdd_plan_set_y_budget")

    def output_shape(self) -> Tuple[int, int]:
        """(floats per TIME row, float2 per FOURIER row) after set_decimation."""
        a, b = ctypes.c_longlong(), ctypes.c_longlong()
        _check(load_library().fdd_plan_get_output_shape(self._h, ctypes.byref(a), ctypes.byref(b)),
               "fdd_plan_get_output_shape")
        return int(a.value), int(b.value)

    def set_profiling(self, enable: bool) -> None:
        _check(load_library().fdd_plan_set_profiling(self._h, int(bool(enable))),
               "fdd_plan_set_profiling")

    def get_stage_ms(self):
        """({stage: ms}, {stage: launches}) of the last execute (needs set_profiling(True))."""
        ms = (ctypes.c_float * FDD_NUM_STAGES)()
        ln = (ctypes.c_int * FDD_NUM_STAGES)()
        _check(load_library().fdd_plan_get_stage_ms(self._h, ms, ln), "fdd_plan_get_stage_ms")
        return ({n: float(ms[i]) for i, n in enumerate(STAGE_NAMES)},
                {n: int(ln[i]) for i, n in enumerate(STAGE_NAMES)})

    def get_spectrum(self) -> Tuple[int, int, float]:
        """(device pointer, row pitch in float2 elements, DC removed per channel) of X[nchans][pitch]."""
        x, pitch, dc = ctypes.c_void_p(), ctypes.c_longlong(), ctypes.c_double()
        _check(load_library().fdd_plan_get_spectrum(self._h, ctypes.byref(x), ctypes.byref(pitch),
                                                    ctypes.byref(dc)), "fdd_plan_get_spectrum")
        return x.value, pitch.value, dc.value

    def get_inverse(self) -> int:
        """The inverse transform the last TIME-mode prepare / execute used (FDD_INVERSE_TWO_PASS or _CUFFT)."""
        w = ctypes.c_int()
        _check(load_library().fdd_plan_get_inverse(self._h, ctypes.byref(w)), "fdd_plan_get_inverse")
        return int(w.value)

    def get_padding(self) -> int:
        """Lowest bins whose mean-rectangle term a per-plan fp64 table supplies (0: not zero padded)."""
        n = ctypes.c_longlong()
        _check(load_library().fdd_plan_get_padding(self._h, ctypes.byref(n)), "fdd_plan_get_padding")
        return int(n.value)

    def destroy(self) -> None:
        if self._h is not None and self._h.value:
            load_library().fdd_plan_destroy(self._h)
        self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()


def measure_fp32_peak(packed: bool, iters: int = 4096) -> Tuple[float, float]:
    """(TFLOP/s, ms) of the register-resident FMA probe on the current device."""
    tf, ms = ctypes.c_double(), ctypes.c_float()
    _check(load_library().fdd_measure_fp32_peak(int(bool(packed)), int(iters), ctypes.byref(tf),
                                                ctypes.byref(ms)), "fdd_measure_fp32_peak")
    return tf.value, ms.value


def tc_selftest(a_f16, b_f16, d_out, stream=None) -> None:
    """d_out[128][64] f32 = a_f16[128][64] @ b_f16[64][64].T on the tcgen05 path (device tensors)."""
    _check(load_library().fdd_tc_selftest(_ptr(a_f16), _ptr(b_f16), _ptr(d_out), _stream_handle(stream)),
           "fdd_tc_selftest")


def rotate_sum_static(x_dev, xpitch: int, delays_dev, nchans: int, nbins: int, nfft: int, ndm: int, out_dev,
                      dc_add: float = 0.0, stream=None) -> None:
    """Step a4 without any allocation (scratch in a static device array of FDD_STATIC_MAX_PHASES entries):
    out_dev[ndm][nbins] c64 = sum over channels of x_dev[nchans][xpitch] c64 rotated by delays_dev[ndm][nchans]
    f64 (device tensors or addresses).  Calls that overlap on the GPU race: include/fdd.h."""
    _check(load_library().fdd_rotate_sum_static(_ptr(x_dev), int(xpitch), _ptr(delays_dev), int(nchans), int(nbins),
                                                int(nfft), int(ndm), _ptr(out_dev), float(dc_add),
                                                _stream_handle(stream)), "fdd_rotate_sum_static")

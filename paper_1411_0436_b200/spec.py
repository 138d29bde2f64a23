"""ctypes binding of include/spec.h — argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; this module holds no
arithmetic and has no CPU fallback: importing it without the built library raises.
PyTorch (if the caller uses it) only supplies device memory (`tensor.data_ptr()`) and streams
(`torch.cuda.current_stream().cuda_stream`); this module itself does not import torch.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libspec.so")

MODE_PFB, MODE_FFT = 0, 1
WINDOW_RECT, WINDOW_HANN = 0, 1
OPT_TENSOR_CORE_STAGE = 1
OK, ERR_ARG, ERR_STATE, ERR_SIZE, ERR_OVERRUN, ERR_CUDA, ERR_NOMEM = 0, -1, -2, -3, -4, -5, -6

# every symbol include/spec.h declares (tests check the library exports all of them)
SYMBOLS = [
    "spec_create", "spec_set_coeffs", "spec_process", "spec_read_accum", "spec_destroy",
    "spec_pending", "spec_spectra_done", "spec_reset", "spec_set_ring", "spec_get_coeffs",
    "spec_stream_host", "spec_measure_fp32_peak", "spec_debug_unpack", "spec_debug_fir",
    "spec_strerror", "spec_last_error", "spec_profile", "spec_profile_read", "spec_read_accum_batch",
    "spec_plan_info", "spec_debug_hog", "spec_set_option", "spec_capture_begin", "spec_capture_end", "spec_replayed",
    "spec_accumulate_host", "spec_create_subbands", "spec_debug_probe", "spec_oneshot_static",
]

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python -m paper_1411_0436_b200.build` "
        "(there is no CPU fallback)")

_lib = C.CDLL(LIB_PATH)
_vp, _sz, _fp = C.c_void_p, C.c_size_t, C.POINTER(C.c_float)
_lib.spec_create.argtypes = [C.POINTER(_vp), C.c_int, C.c_int, C.c_int, C.c_int, C.c_long, C.c_int]
_lib.spec_create_subbands.argtypes = [C.POINTER(_vp), C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_long, C.c_int]
_lib.spec_set_coeffs.argtypes = [_vp, _fp, _sz]
_lib.spec_process.argtypes = [_vp, _vp, _sz, _vp]
_lib.spec_read_accum.argtypes = [_vp, _vp, C.c_int, _vp]
_lib.spec_read_accum_batch.argtypes = [_vp, _vp, C.c_int, _vp]
_lib.spec_destroy.argtypes = [_vp]
_lib.spec_pending.argtypes = [_vp]
_lib.spec_spectra_done.argtypes = [_vp]
_lib.spec_spectra_done.restype = C.c_long
_lib.spec_reset.argtypes = [_vp]
_lib.spec_set_ring.argtypes = [_vp, C.c_int]
_lib.spec_get_coeffs.argtypes = [_vp, _fp, _sz]
_lib.spec_stream_host.argtypes = [_vp, _vp, _sz, _sz, _vp]
_lib.spec_measure_fp32_peak.argtypes = [C.POINTER(C.c_double), _vp]
_lib.spec_debug_unpack.argtypes = [_vp, _sz, C.c_int, _vp, _vp]
_lib.spec_debug_fir.argtypes = [_vp, _vp, C.c_int, _vp, _vp]
_lib.spec_debug_hog.argtypes = [C.c_int, _sz, _vp]
_lib.spec_oneshot_static.argtypes = [_vp, _sz, C.c_int, C.c_int, C.c_int, _vp, _vp, _vp]
_lib.spec_debug_probe.argtypes = [C.c_int, C.POINTER(C.c_double), _vp]
_lib.spec_set_option.argtypes = [_vp, C.c_int, C.c_int]
_lib.spec_capture_begin.argtypes = [_vp]
_lib.spec_capture_end.argtypes = [_vp]
_lib.spec_replayed.argtypes = [_vp, C.c_long]
_lib.spec_accumulate_host.argtypes = [C.POINTER(C.c_double), _fp, _sz]
_lib.spec_plan_info.argtypes = [_vp, C.POINTER(C.c_int), C.POINTER(C.c_int), C.c_char_p, _sz]
_lib.spec_profile.argtypes = [_vp, C.c_int]
_lib.spec_profile_read.argtypes = [_vp, C.POINTER(C.c_double), C.POINTER(C.c_long)]
_lib.spec_strerror.argtypes = [C.c_int]
_lib.spec_strerror.restype = C.c_char_p
_lib.spec_last_error.argtypes = []
_lib.spec_last_error.restype = C.c_char_p


class SpecError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        detail = _lib.spec_last_error().decode() if code in (ERR_CUDA, ERR_NOMEM) else ""
        super().__init__(f"{where}: {_lib.spec_strerror(code).decode()} ({code}) {detail}".strip())


def _check(rc, where):
    if rc < 0:
        raise SpecError(rc, where)
    return rc


def strerror(code):
    return _lib.spec_strerror(code).decode()


def measure_fp32_peak(stream=0):
    out = C.c_double(0.0)
    _check(_lib.spec_measure_fp32_peak(C.byref(out), stream), "spec_measure_fp32_peak")
    return out.value


def debug_unpack(d_bytes_ptr, nbytes, d_out_ptr, stream=0, npol=2):
    _check(_lib.spec_debug_unpack(d_bytes_ptr, nbytes, npol, d_out_ptr, stream), "spec_debug_unpack")


PROBES = ("FFMA", "FFMA2", "FADD2", "PRMT", "LDS.128", "LDS.128 with 8 FFMA2 each", "SHFL")


def debug_probe(op, stream=0):
    """Thread-instructions per clock and SM of instruction kind PROBES[op]."""
    out = C.c_double(0.0)
    _check(_lib.spec_debug_probe(op, C.byref(out), stream), "spec_debug_probe")
    return out.value


def oneshot_static(d_in_ptr, nsamples, nchan, d_out_ptr, ntaps=1, npol=2, d_coeffs_ptr=None, stream=0):
    """spec_oneshot_static: the chain over one stretch of samples with no handle and no allocation; returns the spectra summed."""
    rc = _lib.spec_oneshot_static(d_in_ptr, nsamples, nchan, ntaps, npol, d_coeffs_ptr, d_out_ptr, stream)
    if rc == ERR_SIZE and nchan > 4096:      # the library says which limit was exceeded
        e = SpecError(rc, "spec_oneshot_static")
        e.args = (f"{e.args[0]} {_lib.spec_last_error().decode()}",)
        raise e
    return _check(rc, "spec_oneshot_static")


def debug_hog(ms, smem_bytes, stream=0):
    _check(_lib.spec_debug_hog(ms, smem_bytes, stream), "spec_debug_hog")


def accumulate_host(h_acc, h_spectrum):
    """h_acc (float64, C-contiguous) += h_spectrum (float32), in the library (the CPU thread)."""
    assert h_acc.dtype == np.float64 and h_spectrum.dtype == np.float32 and h_acc.size == h_spectrum.size
    assert h_acc.flags.c_contiguous and h_spectrum.flags.c_contiguous
    _check(_lib.spec_accumulate_host(h_acc.ctypes.data_as(C.POINTER(C.c_double)), h_spectrum.ctypes.data_as(_fp),
                                     h_acc.size), "spec_accumulate_host")


class Spec:
    """Thin handle around spec_t*.  Pointers are integers (device or host addresses)."""

    def __init__(self, nchan, ntaps, npol, mode, nacc, window=WINDOW_HANN, nsub=1):
        h = _vp()
        if nsub == 1:
            _check(_lib.spec_create(C.byref(h), nchan, ntaps, npol, mode, nacc, window), "spec_create")
        else:
            _check(_lib.spec_create_subbands(C.byref(h), nsub, nchan, ntaps, npol, mode, nacc, window),
                   "spec_create_subbands")
        self._h = h
        self.nsub = nsub
        self.nchan, self.npol, self.mode, self.nacc = nchan, npol, mode, nacc
        self.ntaps = 1 if mode == MODE_FFT else ntaps
        self.nstokes = 4 if npol == 2 else 1
        self.ncoef = nchan * self.ntaps

    def set_coeffs(self, h):
        h = np.ascontiguousarray(h, dtype=np.float32).reshape(-1)
        _check(_lib.spec_set_coeffs(self._h, h.ctypes.data_as(_fp), h.size), "spec_set_coeffs")

    def get_coeffs(self):
        out = np.empty(self.ncoef, dtype=np.float32)
        _check(_lib.spec_get_coeffs(self._h, out.ctypes.data_as(_fp), out.size), "spec_get_coeffs")
        return out

    def process(self, d_in_ptr, nsamples, stream=0):
        return _check(_lib.spec_process(self._h, d_in_ptr, nsamples, stream), "spec_process")

    def read_accum_device(self, d_dst_ptr, stream=0):
        return _check(_lib.spec_read_accum(self._h, d_dst_ptr, 1, stream), "spec_read_accum")

    def read_accum_batch_device(self, d_dst_ptr, max_count, stream=0):
        """Pops up to max_count accumulations into device memory [count][S][nchan]; returns the count."""
        return _check(_lib.spec_read_accum_batch(self._h, d_dst_ptr, max_count, stream), "spec_read_accum_batch")

    def read_accum_host(self, stream=0):
        shape = (self.nstokes, self.nchan) if self.nsub == 1 else (self.nsub, self.nstokes, self.nchan)
        out = np.empty(shape, dtype=np.float32)
        rc = _check(_lib.spec_read_accum(self._h, out.ctypes.data, 0, stream), "spec_read_accum")
        return out if rc == 1 else None

    def stream_host(self, h_pinned_ptr, nsamples, chunk_samples, stream=0):
        return _check(_lib.spec_stream_host(self._h, h_pinned_ptr, nsamples, chunk_samples, stream),
                      "spec_stream_host")

    def pending(self):
        return _check(_lib.spec_pending(self._h), "spec_pending")

    def spectra_done(self):
        return _lib.spec_spectra_done(self._h)

    def reset(self):
        _check(_lib.spec_reset(self._h), "spec_reset")

    def set_option(self, option, value):
        _check(_lib.spec_set_option(self._h, option, value), "spec_set_option")

    def capture_begin(self):
        _check(_lib.spec_capture_begin(self._h), "spec_capture_begin")

    def capture_end(self):
        _check(_lib.spec_capture_end(self._h), "spec_capture_end")

    def replayed(self, times):
        _check(_lib.spec_replayed(self._h, times), "spec_replayed")

    def set_ring(self, nslots):
        _check(_lib.spec_set_ring(self._h, nslots), "spec_set_ring")

    def profile(self, enable=True):
        _check(_lib.spec_profile(self._h, 1 if enable else 0), "spec_profile")

    def profile_read(self):
        """{class: (ms, launches)} for classes single, passA, passB, readout."""
        ms = (C.c_double * 4)()
        n = (C.c_long * 4)()
        _check(_lib.spec_profile_read(self._h, ms, n), "spec_profile_read")
        return {k: (ms[i], n[i]) for i, k in enumerate(("single", "passA", "passB", "readout"))}

    def debug_fir(self, d_blocks_ptr, d_out_ptr, stream=0, nspec=1):
        _check(_lib.spec_debug_fir(self._h, d_blocks_ptr, nspec, d_out_ptr, stream), "spec_debug_fir")

    def plan_info(self):
        """(n1, n2, description) of the kernels this handle's plan uses."""
        n1, n2 = C.c_int(0), C.c_int(0)
        buf = C.create_string_buffer(512)
        _check(_lib.spec_plan_info(self._h, C.byref(n1), C.byref(n2), buf, len(buf)), "spec_plan_info")
        return n1.value, n2.value, buf.value.decode()

    def close(self):
        if getattr(self, "_h", None):
            _lib.spec_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

"""CPU ORACLE binding — TEST INFRASTRUCTURE, not the product.

ctypes wrapper over oracle/spec_oracle.c (plain C, double precision; see spec_oracle.h for
the passages of PAPER.md each function follows).  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It imports nothing
from paper_1411_0436_b200 and shares no code with the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "spec_oracle.c")
_LIB = os.path.join(_HERE, "libspec_oracle.so")

MODE_PFB, MODE_FFT = 0, 1
WINDOW_RECT, WINDOW_HANN = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(
        os.path.getmtime(_SRC), os.path.getmtime(os.path.join(_HERE, "spec_oracle.h"))
    ):
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-Wall", "-Wextra", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        )
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        fp = C.POINTER(C.c_float)
        L.oracle_default_coeffs.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, fp]
        L.oracle_default_coeffs.restype = None
        L.oracle_fir.argtypes = [C.c_int, C.c_int, dp, dp, dp]
        L.oracle_fir.restype = None
        for f in (L.oracle_dft_bruteforce, L.oracle_fft_radix2, L.oracle_dft):
            f.argtypes = [C.c_int, dp, dp]
            f.restype = None
        L.oracle_unpack.argtypes = [C.c_int8]
        L.oracle_unpack.restype = C.c_double
        L.oracle_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_long, C.c_int]
        L.oracle_create.restype = C.c_void_p
        L.oracle_set_coeffs.argtypes = [C.c_void_p, fp, C.c_size_t]
        L.oracle_set_coeffs.restype = C.c_int
        L.oracle_process.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
        L.oracle_process.restype = C.c_long
        L.oracle_read_accum.argtypes = [C.c_void_p, dp]
        L.oracle_read_accum.restype = C.c_int
        L.oracle_pending.argtypes = [C.c_void_p]
        L.oracle_pending.restype = C.c_long
        L.oracle_spectra_done.argtypes = [C.c_void_p]
        L.oracle_spectra_done.restype = C.c_long
        L.oracle_reset.argtypes = [C.c_void_p]
        L.oracle_reset.restype = None
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_destroy.restype = None
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def default_coeffs(nchan, ntaps, mode=MODE_PFB, window=WINDOW_HANN):
    n = nchan if mode == MODE_FFT else nchan * ntaps
    out = np.empty(n, dtype=np.float32)
    lib().oracle_default_coeffs(nchan, ntaps, mode, window, out.ctypes.data_as(C.POINTER(C.c_float)))
    return out


def _cplx_io(fn, n, x):
    x = np.ascontiguousarray(x, dtype=np.complex128)
    assert x.shape == (n,)
    out = np.empty(n, dtype=np.complex128)
    fn(n, _dp(x.view(np.float64)), _dp(out.view(np.float64)))
    return out


def dft_bruteforce(x):
    return _cplx_io(lib().oracle_dft_bruteforce, len(x), x)


def fft_radix2(x):
    return _cplx_io(lib().oracle_fft_radix2, len(x), x)


def dft(x):
    return _cplx_io(lib().oracle_dft, len(x), x)


def fir(h, x, nchan, ntaps):
    """h: T*N real; x: T*N complex (T blocks); returns N complex."""
    h = np.ascontiguousarray(h, dtype=np.float64)
    x = np.ascontiguousarray(x, dtype=np.complex128)
    assert h.shape == (nchan * ntaps,) and x.shape == (nchan * ntaps,)
    y = np.empty(nchan, dtype=np.complex128)
    lib().oracle_fir(nchan, ntaps, _dp(h), _dp(x.view(np.float64)), _dp(y.view(np.float64)))
    return y


def unpack(b):
    return lib().oracle_unpack(int(b))


class Oracle:
    """Streaming state machine (PAPER.md:87-96 steps 1-7)."""

    def __init__(self, nchan, ntaps, npol, mode, nacc, window=WINDOW_HANN):
        self._h = lib().oracle_create(nchan, ntaps, npol, mode, nacc, window)
        if not self._h:
            raise ValueError("oracle_create: bad arguments")
        self.nchan, self.npol = nchan, npol
        self.ntaps = 1 if mode == MODE_FFT else ntaps
        self.nstokes = 4 if npol == 2 else 1

    def set_coeffs(self, h):
        h = np.ascontiguousarray(h, dtype=np.float32)
        if lib().oracle_set_coeffs(self._h, h.ctypes.data_as(C.POINTER(C.c_float)), h.size) != 0:
            raise ValueError("oracle_set_coeffs: wrong count")

    def process(self, raw):
        """raw: int8 array, 2*npol bytes per time sample."""
        raw = np.ascontiguousarray(raw, dtype=np.int8).reshape(-1)
        ns, rem = divmod(raw.size, 2 * self.npol)
        if rem:
            raise ValueError("partial sample")
        r = lib().oracle_process(self._h, raw.ctypes.data, ns)
        if r < 0:
            raise ValueError("oracle_process: nsamples not a multiple of nchan")
        return r

    def read_accum(self):
        out = np.empty((self.nstokes, self.nchan), dtype=np.float64)
        return out if lib().oracle_read_accum(self._h, _dp(out)) == 1 else None

    def pending(self):
        return lib().oracle_pending(self._h)

    def spectra_done(self):
        return lib().oracle_spectra_done(self._h)

    def reset(self):
        lib().oracle_reset(self._h)

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class OracleSub:
    """Eight-sub-band modes (PAPER.md:51, :73 Table 1 third block, :90 step 1b "16 FFTs in parallel"): nsub
    independent spectrometers that share channel count, filter and accumulation length.  Reading (R26;
    the paper does not state the order): the sub-bands are interleaved per time sample, sub-band 0 first, i.e. the
    byte stream is [time sample][sub-band][2*npol bytes].  The oracle is that definition written out: take every
    nsub-th word and run the single-sub-band state machine on it."""

    def __init__(self, nsub, nchan, ntaps, npol, mode, nacc, window=WINDOW_HANN):
        self.nsub, self.npol = nsub, npol
        self.subs = [Oracle(nchan, ntaps, npol, mode, nacc, window) for _ in range(nsub)]

    def set_coeffs(self, h):
        for o in self.subs:
            o.set_coeffs(h)

    def process(self, raw):
        raw = np.ascontiguousarray(raw, dtype=np.int8).reshape(-1, self.nsub, 2 * self.npol)
        r = 0
        for s, o in enumerate(self.subs):
            r = o.process(np.ascontiguousarray(raw[:, s, :]))
        return r

    def read_accum(self):
        outs = [o.read_accum() for o in self.subs]
        return None if outs[0] is None else np.stack(outs)

    def pending(self):
        return self.subs[0].pending()

    def spectra_done(self):
        return self.subs[0].spectra_done()

    def close(self):
        for o in self.subs:
            o.close()

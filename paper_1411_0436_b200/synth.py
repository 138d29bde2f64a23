"""Seeded synthetic input streams (shared by the oracle tests, the GPU parity tests and bench.py).

This module holds NONE of the method's arithmetic (no unpack, FIR, FFT or Stokes): it only
draws the int8 sample streams BASELINE.json's configs describe.  The paper's own benchmark
inputs were disk files pre-loaded in memory (section 5) and are not available;
these streams stand in for them with the shapes of Table 1.  numpy only.

Recipe:
  * noise: independent N(0, sigma^2) per real/imaginary component, numpy default_rng;
  * tone:  A * exp(+2 pi i f j), j = absolute sample index from 0, phase 0, f = num/den
           cycles per sample held as an exact rational so the phase is exact at any j;
  * quantisation: round-half-to-even (np.rint), clip to [-127, 127], int8;
  * the stream is generated in fixed chunks of 2**20 samples, chunk c seeded with
    (seed, c), so any [start, start+n) slice is reproducible however callers split it.
Byte layout per time sample (BASELINE.json configs): dual-pol [Xre, Xim, Yre, Yim],
single-pol [re, im].
"""
from __future__ import annotations

from fractions import Fraction

import numpy as np

SEED_BASE = 14110436
_CHUNK = 1 << 20


def _tone(amp, freq: Fraction, j0: int, n: int):
    j = np.arange(j0, j0 + n, dtype=np.int64)
    num, den = freq.numerator, freq.denominator
    ph = ((j * (num % den)) % den).astype(np.float64) / float(den)  # exact fractional cycles
    return amp * np.exp(2j * np.pi * ph)


def _quant(z):
    out = np.empty(z.shape + (2,), dtype=np.int8)
    out[..., 0] = np.clip(np.rint(z.real), -127, 127).astype(np.int8)
    out[..., 1] = np.clip(np.rint(z.imag), -127, 127).astype(np.int8)
    return out


def _chunks(start, n):
    c0, c1 = start // _CHUNK, (start + n - 1) // _CHUNK
    for c in range(c0, c1 + 1):
        lo = max(start, c * _CHUNK)
        hi = min(start + n, (c + 1) * _CHUNK)
        yield c, lo - c * _CHUNK, hi - c * _CHUNK


def single_pol_stream(seed, nsamples, tones, sigma=16.0, amp=20.0, start=0):
    """int8 [nsamples, 2] = (re, im).  tones: list of Fraction cycles/sample."""
    out = np.empty((nsamples, 2), dtype=np.int8)
    pos = 0
    for c, lo, hi in _chunks(start, nsamples):
        rng = np.random.default_rng([seed, c])
        g = rng.standard_normal((_CHUNK, 2))
        z = sigma * (g[lo:hi, 0] + 1j * g[lo:hi, 1])
        for f in tones:
            z = z + _tone(amp, Fraction(f), c * _CHUNK + lo, hi - lo)
        out[pos:pos + hi - lo] = _quant(z)
        pos += hi - lo
    return out


def dual_pol_stream(seed, nsamples, tones, sigma=12.0, amp=20.0, start=0):
    """Config-1 generator: X = s + n1, Y = 0.7 s e^{i pi/5} + n2, tones added to s.
    Returns int8 [nsamples, 4] = (Xre, Xim, Yre, Yim)."""
    out = np.empty((nsamples, 4), dtype=np.int8)
    rot = 0.7 * np.exp(1j * np.pi / 5.0)
    pos = 0
    for c, lo, hi in _chunks(start, nsamples):
        rng = np.random.default_rng([seed, c])
        g = rng.standard_normal((_CHUNK, 6))[lo:hi]
        s = sigma * (g[:, 0] + 1j * g[:, 1])
        n1 = sigma * (g[:, 2] + 1j * g[:, 3])
        n2 = sigma * (g[:, 4] + 1j * g[:, 5])
        for f in tones:
            s = s + _tone(amp, Fraction(f), c * _CHUNK + lo, hi - lo)
        x = s + n1
        y = rot * s + n2
        n = hi - lo
        out[pos:pos + n, 0:2] = _quant(x)
        out[pos:pos + n, 2:4] = _quant(y)
        pos += n
    return out


# ---------------------------------------------------------------- BASELINE.json configs

CONFIGS = {
    0: dict(name="cfg0_pfb_1k_singlepol", mode="pfb", nchan=1024, ntaps=8, npol=1, nacc=64,
            nsamples=(64 + 7) * 1024, calls=1),
    1: dict(name="cfg1_pfb_32k_dualpol", mode="pfb", nchan=32768, ntaps=8, npol=2, nacc=256,
            nsamples=4 * (1 << 24), calls=4),  # 4 calls x 64 MiB (reading R14)
    2: dict(name="cfg2_fft_4k_dualpol", mode="fft", nchan=4096, ntaps=1, npol=2, nacc=2048,
            nsamples=2048 * 4096, calls=1),
    3: dict(name="cfg3_pfb_512k_dualpol", mode="pfb", nchan=524288, ntaps=8, npol=2, nacc=16,
            nsamples=(16 + 7) * 524288, calls=1),
}

F_CFG1 = Fraction(20001, 131072)  # 5000.25 / 32768 cycles per sample


def config_stream(cfg: int, start=0, nsamples=None):
    """The int8 stream of config `cfg` (slice [start, start+nsamples))."""
    c = CONFIGS[cfg]
    n = c["nsamples"] - start if nsamples is None else nsamples
    seed = SEED_BASE + cfg
    if cfg == 0:
        N = c["nchan"]
        return single_pol_stream(seed, n, [Fraction(100, N), Fraction(601, 2 * N)], start=start)
    if cfg in (1, 2):
        return dual_pol_stream(seed, n, [F_CFG1], start=start)
    if cfg == 3:
        N = c["nchan"]
        return dual_pol_stream(seed, n, [Fraction(1000, N), Fraction(524289, 2 * N)], start=start)
    raise KeyError(cfg)


def random_bytes(seed, nsamples, npol):
    """Uniform int8 over the full range [-128, 127] (edge-case streams)."""
    rng = np.random.default_rng(seed)
    return rng.integers(-128, 128, size=(nsamples, 2 * npol), dtype=np.int8)


def random_coeffs(seed, count):
    """Arbitrary fp32 coefficient array for spec_set_coeffs tests (an input, not the prototype filter)."""
    rng = np.random.default_rng(seed)
    return rng.uniform(-1.0, 1.0, size=count).astype(np.float32)

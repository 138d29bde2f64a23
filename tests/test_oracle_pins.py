"""Pins for the CPU oracle (oracle/spec_oracle.c) — CPU only, no GPU, no CUDA library.

Each test checks the oracle against something other than itself: a closed form, an invariant,
a library routine (numpy.fft), brute force on a tiny input written in a different form, or a
value stored under tests/golden/ with its citation.  Chosen so that a dropped term, a wrong
sign or index, a transposed operand or a wrong byte lane fails at least one of them.
Citations are PAPER.md lines (section 4 unless noted) and SURVEY.md section 8(c) rows.
"""
import json
import os

import numpy as np
import pytest

import oracle
from oracle import MODE_FFT, MODE_PFB, WINDOW_HANN, WINDOW_RECT, Oracle
from paper_1411_0436_b200 import synth

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "pfb_pins.json")))
T8 = 8


# ---------------------------------------------------------------- unpack (A14)

def test_unpack_all_256_values():
    for v in range(-128, 128):
        assert oracle.unpack(v) == float(v)


# ---------------------------------------------------------------- DFT (A5, A6)

@pytest.mark.parametrize("fn", [oracle.dft_bruteforce, oracle.fft_radix2, oracle.dft])
@pytest.mark.parametrize("n", [1, 2, 8, 64, 256, 512])
def test_dft_of_delta_is_phase_ramp(fn, n):
    # delta at j0 -> X[k] = exp(-2 pi i j0 k / n): fixes sign and absence of scaling
    j0 = 3 % n
    x = np.zeros(n, complex)
    x[j0] = 1.0
    X = fn(x)
    k = np.arange(n)
    np.testing.assert_allclose(X, np.exp(-2j * np.pi * j0 * k / n), atol=1e-12)


@pytest.mark.parametrize("fn", [oracle.dft_bruteforce, oracle.fft_radix2])
@pytest.mark.parametrize("n,c", [(16, 5), (256, 100), (512, 300)])
def test_positive_tone_peaks_at_its_channel(fn, n, c):
    # A5: A e^{+2 pi i c j/N} -> N*A at index c (not N-c), zero elsewhere; A6: unnormalised
    j = np.arange(n)
    X = fn(2.5 * np.exp(2j * np.pi * c * j / n))
    want = np.zeros(n, complex)
    want[c] = 2.5 * n
    np.testing.assert_allclose(X, want, atol=1e-9 * n)


def test_bruteforce_any_length_matches_numpy():
    rng = np.random.default_rng(1)
    for n in (1, 2, 3, 5, 12, 64, 255, 256):
        x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
        np.testing.assert_allclose(oracle.dft_bruteforce(x), np.fft.fft(x), rtol=0, atol=1e-10 * n)


@pytest.mark.parametrize("n", [2, 4, 256, 512, 1024, 4096, 32768])
def test_radix2_matches_numpy(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    X = oracle.fft_radix2(x)
    ref = np.fft.fft(x)
    assert np.linalg.norm(X - ref) / np.linalg.norm(ref) < 1e-13


@pytest.mark.parametrize("n", [256, 512])
def test_bruteforce_vs_radix2_at_switch_over(n):
    rng = np.random.default_rng(7)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    a, b = oracle.dft_bruteforce(x), oracle.fft_radix2(x)
    assert np.linalg.norm(a - b) / np.linalg.norm(a) < 1e-12
    # oracle.dft picks brute force up to 256 and radix-2 above (north_star)
    np.testing.assert_array_equal(oracle.dft(x), a if n <= 256 else b)


def test_shift_theorem_and_linearity():
    rng = np.random.default_rng(3)
    n = 512
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    y = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    X, Y = oracle.fft_radix2(x), oracle.fft_radix2(y)
    k = np.arange(n)
    np.testing.assert_allclose(oracle.fft_radix2(np.roll(x, 1)), X * np.exp(-2j * np.pi * k / n), atol=1e-10)
    np.testing.assert_allclose(oracle.fft_radix2(2 * x - 3j * y), 2 * X - 3j * Y, atol=1e-9)


# ---------------------------------------------------------------- coefficients (A1, golden)

@pytest.mark.parametrize("n", [64, 1024, 32768])
def test_sinc_hann_prototype_pins(n):
    h = oracle.default_coeffs(n, T8, MODE_PFB, WINDOW_HANN).astype(np.float64)
    L = T8 * n
    assert h.shape == (L,)
    assert h[0] == 0.0
    assert h[L // 2] == 1.0
    np.testing.assert_allclose(h[1:], h[1:][::-1], atol=1e-7)  # h[k] = h[TN-k]
    # zeros of the sinc at multiples of N away from the centre
    for t in range(T8):
        if t != T8 // 2:
            assert abs(h[t * n]) < 1e-7
    if n >= 1024:
        np.testing.assert_allclose(h.sum() / n, GOLD["sum_h_over_N"], rtol=2e-7)
        np.testing.assert_allclose((h * h).sum() / n, GOLD["sum_h2_over_N"], rtol=2e-7)
        g = h.reshape(T8, n).sum(axis=0)
        assert abs(g.min() - GOLD["branch_gain_min"]) < 2e-6
        assert abs(g.max() - GOLD["branch_gain_max"]) < 2e-6


def test_rect_and_fft_mode_coefficients():
    n = 256
    np.testing.assert_array_equal(oracle.default_coeffs(n, 1, MODE_FFT, WINDOW_RECT), np.ones(n, np.float32))
    w = oracle.default_coeffs(n, 1, MODE_FFT, WINDOW_HANN).astype(np.float64)
    np.testing.assert_allclose(w, np.hanning(n + 1)[:-1], atol=1e-7)  # periodic Hann = symmetric of n+1 minus last
    h = oracle.default_coeffs(n, 4, MODE_PFB, WINDOW_RECT).astype(np.float64)
    k = np.arange(4 * n)
    np.testing.assert_allclose(h, np.sinc((k - 2 * n) / n), atol=1e-7)


# ---------------------------------------------------------------- FIR (A2)

def test_fir_single_tap_selects_that_block():
    n, t = 32, 5
    rng = np.random.default_rng(2)
    x = rng.standard_normal(n * t) + 1j * rng.standard_normal(n * t)
    for sel in range(t):
        h = np.zeros(n * t)
        h[sel * n:(sel + 1) * n] = 1.0
        np.testing.assert_array_equal(oracle.fir(h, x, n, t), x[sel * n:(sel + 1) * n])


def test_fir_matches_einsum():
    n, t = 48, 8
    rng = np.random.default_rng(4)
    x = rng.standard_normal(n * t) + 1j * rng.standard_normal(n * t)
    h = rng.standard_normal(n * t)
    ref = np.einsum("tn,tn->n", h.reshape(t, n), x.reshape(t, n))
    np.testing.assert_allclose(oracle.fir(h, x, n, t), ref, atol=1e-12)


@pytest.mark.parametrize("n,n0", [(64, 0), (64, 17), (512, 300)])
def test_impulse_reproduces_coefficients(n, n0):
    """north_star / A2: an impulse at j0=(T-1)N+n0 gives |X_m[k]|^2 = h[(T-1-m)N+n0]^2 flat in k,
    for m = 0..T-1 (taps appear in reverse order over m)."""
    T = T8
    h = oracle.default_coeffs(n, T, MODE_PFB, WINDOW_HANN).astype(np.float64)
    raw = np.zeros(((2 * T - 1) * n, 2), np.int8)
    raw[(T - 1) * n + n0, 0] = 1
    o = Oracle(n, T, 1, MODE_PFB, 1)
    assert o.process(raw) == T
    for m in range(T):
        out = o.read_accum()
        want = h[(T - 1 - m) * n + n0] ** 2
        np.testing.assert_allclose(out[0], np.full(n, want), atol=1e-12)
    assert o.read_accum() is None


# ---------------------------------------------------------------- PFB response (A6, A7, A8)

def _pfb_spectrum(n, f_chan, amp=20.0):
    h = oracle.default_coeffs(n, T8, MODE_PFB, WINDOW_HANN).astype(np.float64)
    j = np.arange(T8 * n)
    x = amp * np.exp(2j * np.pi * f_chan * j / n)
    return h, oracle.dft(oracle.fir(h, x, n, T8))


@pytest.mark.parametrize("n", [256, 1024])
def test_integer_channel_tone_containment_and_gain(n):
    c = 100
    h, X = _pfb_spectrum(n, c)
    p = np.abs(X) ** 2
    frac = p[c] / p.sum()
    assert frac > 0.99  # north_star
    assert abs(frac - GOLD["tone_containment_integer_channel"]) < 2e-8
    np.testing.assert_allclose(p[c], (20.0 * h.sum()) ** 2, rtol=1e-10)  # A6
    if n == 1024:
        np.testing.assert_allclose(p[c], GOLD["cfg0_tone_channel_power_per_spectrum_A20_N1024"], rtol=1e-4)
    np.testing.assert_allclose(p[c + 1] / p[c], GOLD["adjacent_channel_leak_offset_1p0"], rtol=5e-3)


@pytest.mark.parametrize("n", [256, 1024])
def test_half_channel_scalloping(n):
    c = 300 % n
    _, X0 = _pfb_spectrum(n, c)
    _, Xh = _pfb_spectrum(n, c + 0.5)
    p0, ph = np.abs(X0) ** 2, np.abs(Xh) ** 2
    for nb in (c, c + 1):
        assert abs(ph[nb] / p0[c] - GOLD["pfb_half_channel_power_ratio"]) < 2e-6
    assert abs((ph[c] + ph[c + 1]) / ph.sum() - GOLD["pfb_half_channel_two_neighbours_fraction"]) < 2e-8
    # offset 1.5 channels
    np.testing.assert_allclose(ph[c + 2] / p0[c], GOLD["leak_offset_1p5"], rtol=2e-2)


def test_direct_fft_scalloping_is_4_over_pi_squared():
    n, c = 512, 37
    j = np.arange(n)
    p0 = np.abs(oracle.dft(np.exp(2j * np.pi * c * j / n))) ** 2
    ph = np.abs(oracle.dft(np.exp(2j * np.pi * (c + 0.5) * j / n))) ** 2
    # rectangular window: |sin(pi/2)/(N sin(pi/(2N)))|^2 -> sinc^2(1/2) = 4/pi^2 as N grows
    exact = 1.0 / (n * np.sin(np.pi / (2 * n))) ** 2
    np.testing.assert_allclose(ph[c] / p0[c], exact, rtol=1e-10)
    assert abs(ph[c] / p0[c] - 4 / np.pi ** 2) < 1e-5
    assert abs(ph[c] / p0[c] - GOLD["fft_half_channel_power_ratio"]) < 2e-6


def test_parseval_per_spectrum():
    # A9: sum_k |X[k]|^2 = N sum_n |y[n]|^2
    for n in (64, 256, 1024):
        rng = np.random.default_rng(n)
        x = rng.standard_normal(T8 * n) + 1j * rng.standard_normal(T8 * n)
        h = oracle.default_coeffs(n, T8).astype(np.float64)
        y = oracle.fir(h, x, n, T8)
        X = oracle.dft(y)
        np.testing.assert_allclose((np.abs(X) ** 2).sum(), n * (np.abs(y) ** 2).sum(), rtol=1e-12)


# ---------------------------------------------------------------- Stokes (A10-A12)

def test_cross_product_sign_exact():
    """A11: X=1, Y=i in every channel -> Re(XY*)=0, Im(XY*)=-1.  Bytes 01 00 00 01 at sample 0."""
    n = 64
    raw = np.zeros((n, 4), np.int8)
    raw[0] = [1, 0, 0, 1]
    o = Oracle(n, 1, 2, MODE_FFT, 1, WINDOW_RECT)
    assert o.process(raw) == 1
    out = o.read_accum()
    np.testing.assert_array_equal(out[0], np.ones(n))
    np.testing.assert_array_equal(out[1], np.ones(n))
    np.testing.assert_allclose(out[2], np.zeros(n), atol=1e-15)
    np.testing.assert_allclose(out[3], -np.ones(n), atol=1e-15)


def test_stokes_inequalities():
    n, M = 128, 5
    raw = synth.random_bytes(11, (M + T8 - 1) * n, 2)
    o1 = Oracle(n, T8, 2, MODE_PFB, 1)
    oM = Oracle(n, T8, 2, MODE_PFB, M)
    assert o1.process(raw) == M and oM.process(raw) == 1
    acc = np.zeros((4, n))
    for _ in range(M):
        s = o1.read_accum()
        assert (s[0] >= 0).all() and (s[1] >= 0).all()
        # equality at M=1 (Cauchy-Schwarz is tight for a single spectrum)
        np.testing.assert_allclose(s[2] ** 2 + s[3] ** 2, s[0] * s[1], rtol=1e-10)
        acc += s
    S = oM.read_accum()
    np.testing.assert_allclose(S, acc, rtol=1e-13, atol=1e-6)  # A6: accumulate = sum, not mean
    assert (S[2] ** 2 + S[3] ** 2 <= S[0] * S[1] * (1 + 1e-12)).all()
    assert (S[2] ** 2 + S[3] ** 2 < S[0] * S[1]).any()


# ---------------------------------------------------------------- state machine (A3, A4, A13-A16)

def _brute_force_chain(raw, N, T, P, M, h):
    """The whole definition in numpy, written differently from the C code (matrix DFT, einsum)."""
    v = raw.astype(np.float64).reshape(-1, P, 2)
    z = v[..., 0] + 1j * v[..., 1]                      # [sample, pol]
    nblk = z.shape[0] // N
    zb = z.reshape(nblk, N, P)
    F = np.exp(-2j * np.pi * np.outer(np.arange(N), np.arange(N)) / N)
    outs, acc, cnt = [], np.zeros((4 if P == 2 else 1, N)), 0
    for m in range(nblk - T + 1):
        y = np.einsum("tn,tnp->np", h.reshape(T, N), zb[m:m + T])
        X = F.T @ y                                     # [k, pol]
        acc[0] += np.abs(X[:, 0]) ** 2
        if P == 2:
            acc[1] += np.abs(X[:, 1]) ** 2
            c = X[:, 0] * np.conj(X[:, 1])
            acc[2] += c.real
            acc[3] += c.imag
        cnt += 1
        if cnt % M == 0:
            outs.append(acc.copy())
            acc[:] = 0
    return outs


@pytest.mark.parametrize("N,T,P,M,mode", [(8, 3, 2, 2, MODE_PFB), (16, 8, 1, 3, MODE_PFB),
                                          (8, 1, 2, 4, MODE_FFT), (4, 2, 2, 1, MODE_PFB)])
def test_tiny_brute_force(N, T, P, M, mode):
    nblk = 3 * M + T - 1
    raw = synth.random_bytes(100 + N, nblk * N, P)
    h = synth.random_coeffs(5, T * N)
    o = Oracle(N, T, P, mode, M)
    o.set_coeffs(h)
    ref = _brute_force_chain(raw, N, T, P, M, h.astype(np.float64))
    assert o.process(raw) == len(ref) == 3
    for r in ref:
        np.testing.assert_allclose(o.read_accum(), r, rtol=1e-12, atol=1e-9)


def test_spectrum_count_and_empty_start():
    # A3/A4: hop = N, history starts EMPTY: (64+7)*1024 samples -> exactly 64 spectra -> one output
    c = synth.CONFIGS[0]
    o = Oracle(c["nchan"], c["ntaps"], c["npol"], MODE_PFB, c["nacc"])
    assert o.process(np.zeros((c["nsamples"], 2), np.int8)) == 1
    assert o.spectra_done() == 64
    o.reset()
    assert o.process(np.zeros((7 * 1024, 2), np.int8)) == 0 and o.spectra_done() == 0
    assert o.process(np.zeros((1024, 2), np.int8)) == 0 and o.spectra_done() == 1


def test_rejects_partial_block():
    o = Oracle(64, 8, 2, MODE_PFB, 1)
    with pytest.raises(ValueError):
        o.process(np.zeros((65, 4), np.int8))  # A15


def test_split_invariance_is_bit_exact():
    # A16: outputs depend only on the concatenated stream
    N, T, M = 64, 8, 3
    raw = synth.random_bytes(21, 40 * N, 2)
    a = Oracle(N, T, 2, MODE_PFB, M)
    a.process(raw)
    b = Oracle(N, T, 2, MODE_PFB, M)
    cuts = [0, 1, 2, 9, 10, 17, 31, 40]
    total = 0
    for lo, hi in zip(cuts[:-1], cuts[1:]):
        total += b.process(raw[lo * N:hi * N])
    assert total == a.pending() == (40 - 7) // M
    while True:
        x, y = a.read_accum(), b.read_accum()
        if x is None:
            assert y is None
            break
        np.testing.assert_array_equal(x, y)


def test_byte_lanes_and_polarisation_order():
    # A13: [Xre, Xim, Yre, Yim]; a +c tone in X only must land in plane 0 at channel c;
    # swapping re/im sends it to N-c.
    N, c = 64, 5
    j = np.arange(N)
    z = 100 * np.exp(2j * np.pi * c * j / N)
    raw = np.zeros((N, 4), np.int8)
    raw[:, 0] = np.rint(z.real)
    raw[:, 1] = np.rint(z.imag)
    o = Oracle(N, 1, 2, MODE_FFT, 1, WINDOW_RECT)
    o.process(raw)
    s = o.read_accum()
    assert s[0].argmax() == c and s[0][c] / s[0].sum() > 0.999 and s[1].sum() == 0
    o.process(raw[:, [1, 0, 2, 3]])
    assert o.read_accum()[0].argmax() == N - c
    o.process(raw[:, [2, 3, 0, 1]])
    s = o.read_accum()
    assert s[1].argmax() == c and s[0].sum() == 0
    # single-pol layout [re, im]
    o1 = Oracle(N, 1, 1, MODE_FFT, 1, WINDOW_RECT)
    o1.process(raw[:, :2])
    assert o1.read_accum()[0].argmax() == c


def test_minus_128_is_accepted():
    N = 16
    raw = np.full((N, 2), -128, np.int8)
    o = Oracle(N, 1, 1, MODE_FFT, 1, WINDOW_RECT)
    o.process(raw)
    s = o.read_accum()
    np.testing.assert_allclose(s[0][0], (128.0 * N) ** 2 * 2, rtol=1e-14)


def test_fft_mode_ignores_ntaps():
    N = 32
    raw = synth.random_bytes(9, 4 * N, 2)
    a = Oracle(N, 8, 2, MODE_FFT, 4, WINDOW_RECT)
    b = Oracle(N, 1, 2, MODE_FFT, 4, WINDOW_RECT)
    assert a.process(raw) == b.process(raw) == 1
    np.testing.assert_array_equal(a.read_accum(), b.read_accum())


# ---------------------------------------------------------------- generator + oracle end to end

def test_white_noise_gain():
    # A6: mean channel power per spectrum = sigma_tot^2 * sum(h^2) (PFB)
    N, M = 256, 200
    raw = synth.single_pol_stream(5, (M + 7) * N, [], sigma=16.0)
    o = Oracle(N, T8, 1, MODE_PFB, M)
    assert o.process(raw) == 1
    h = oracle.default_coeffs(N, T8).astype(np.float64)
    mean = o.read_accum()[0].mean() / M
    want = (2 * 16.0 ** 2 + 1 / 6) * (h * h).sum()
    assert abs(mean / want - 1) < 0.01


def test_config0_expected_levels():
    """SURVEY 8(c) 'Expected values for config 0': floor ~3.01e7, channel 100 ~2.693e10,
    channels 300 and 301 ~6.71e9 each."""
    c = synth.CONFIGS[0]
    raw = synth.config_stream(0)
    assert raw.shape == (c["nsamples"], 2) and raw.dtype == np.int8
    assert np.abs(raw.astype(int)).max() <= 127
    o = Oracle(c["nchan"], c["ntaps"], 1, MODE_PFB, c["nacc"])
    assert o.process(raw) == 1
    s = o.read_accum()[0]
    quiet = np.delete(s, [99, 100, 101, 299, 300, 301, 302])
    assert abs(np.median(quiet) / 3.01e7 - 1) < 0.08
    assert abs(s[100] / 2.693e10 - 1) < 0.03
    assert abs(s[300] / 6.71e9 - 1) < 0.06 and abs(s[301] / 6.71e9 - 1) < 0.06


def test_config1_cross_phase():
    """A11 (statistical): config-1 generator -> phase of sum_k(Re + i Im) -> -pi/5, |sum XY*|/sum XX -> 0.35."""
    N, M = 256, 64
    raw = synth.dual_pol_stream(synth.SEED_BASE + 1, (M + 7) * N, [])
    o = Oracle(N, T8, 2, MODE_PFB, M)
    o.process(raw)
    s = o.read_accum()
    z = s[2].sum() + 1j * s[3].sum()
    assert abs(np.angle(z) + np.pi / 5) < 0.02
    assert abs(abs(z) / s[0].sum() - 0.35) < 0.01


def test_generator_is_split_invariant():
    a = synth.config_stream(1, 0, 3 * (1 << 20) + 17)
    b = np.concatenate([synth.config_stream(1, 0, (1 << 20) - 5), synth.config_stream(1, (1 << 20) - 5, 2 * (1 << 20) + 22)])
    np.testing.assert_array_equal(a, b)


# ---------------------------------------------------------------- eight-sub-band modes

def test_subband_oracle_places_each_sub_band_in_its_own_output():
    """Reading R26 (sub-bands interleaved per time sample, sub-band 0 first): a tone fed to ONE sub-band shows up
    in that sub-band's output only, at its own channel; the others hold noise-free zeros."""
    N, nsub, M = 64, 8, 4
    j = np.arange(M * N)
    for hot, chan in ((0, 5), (3, 17), (7, 60)):
        raw = np.zeros((M * N, nsub, 4), dtype=np.int8)
        z = 50.0 * np.exp(2j * np.pi * chan * j / N)
        raw[:, hot, 0] = np.rint(z.real)
        raw[:, hot, 1] = np.rint(z.imag)
        o = oracle.OracleSub(nsub, N, 1, 2, oracle.MODE_FFT, M, oracle.WINDOW_RECT)
        assert o.process(raw) == 1
        out = o.read_accum()
        o.close()
        assert out.shape == (nsub, 4, N)
        for s in range(nsub):
            if s == hot:
                assert np.argmax(out[s, 0]) == chan
                assert out[s, 0, chan] > 0.99 * out[s, 0].sum()
            else:
                assert np.all(out[s] == 0)


def test_subband_oracle_equals_the_single_band_oracle_on_every_sub_band():
    """Each sub-band is the single-sub-band chain on its own samples: identical streams in all sub-bands give
    outputs bit-identical to the plain oracle's, and permuting the sub-bands of the input permutes the outputs."""
    N, T, nsub, M = 128, 4, 8, 3
    rng = np.random.default_rng(7)
    base = rng.integers(-128, 128, size=((2 * M + T - 1) * N, 4), dtype=np.int8)
    one = oracle.Oracle(N, T, 2, oracle.MODE_PFB, M)
    one.process(base)
    ref = [one.read_accum(), one.read_accum()]
    one.close()
    raw = np.repeat(base[:, None, :], nsub, axis=1)
    o = oracle.OracleSub(nsub, N, T, 2, oracle.MODE_PFB, M)
    assert o.process(raw) == 2
    for w in range(2):
        out = o.read_accum()
        for s in range(nsub):
            assert np.array_equal(out[s], ref[w])
    o.close()
    # different data per sub-band; a permutation of the sub-bands permutes the outputs
    data = rng.integers(-128, 128, size=((M + T - 1) * N, nsub, 4), dtype=np.int8)
    perm = rng.permutation(nsub)
    a = oracle.OracleSub(nsub, N, T, 2, oracle.MODE_PFB, M)
    b = oracle.OracleSub(nsub, N, T, 2, oracle.MODE_PFB, M)
    a.process(data)
    b.process(data[:, perm, :])
    oa, ob = a.read_accum(), b.read_accum()
    a.close(); b.close()
    assert np.array_equal(ob, oa[perm])
    assert not np.array_equal(oa[0], oa[1])

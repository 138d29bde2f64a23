"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle on the same seeded
inputs.  Bit-exact for the unpack and indexing stages, BASELINE.json north_star tolerances for the
accumulated spectra (tests/_harness.py)."""
import numpy as np
import pytest

from _harness import check_stokes_invariants, compare, gpu_run, make_stream_file, oracle_many, oracle_run
from paper_1411_0436_b200 import synth

pytestmark = pytest.mark.gpu

PFB, FFT = 0, 1


def _torch():
    import torch
    return torch


def _sp():
    from paper_1411_0436_b200 import spec as sp
    return sp


# ---------------------------------------------------------------- bit-exact stages
# north_star: "The unpack and indexing stages must be bit-exact."  spec_debug_fir runs the FRONT END of the
# very kernel the handle's plan uses (a DUMP instantiation of the same template: k_engine, k_fused's
# producers, k_passA_pfb16, k_fir8), so these tests go through the hot path's own staging, index
# arithmetic, unpack and FIR code, not through a stand-in.

@pytest.mark.parametrize("npol", [1, 2])
def test_unpack_bit_exact_all_values_all_lanes(npol):
    torch, sp = _torch(), _sp()
    # every byte value in every byte lane of a 32-bit word, plus a ragged tail (1027 bytes)
    vals = np.arange(-128, 128, dtype=np.int8)
    b = np.concatenate([np.roll(vals, k) for k in range(4)] + [vals[:3]]).astype(np.int8)
    d = torch.from_numpy(b).cuda()
    out = torch.full((b.size,), 1e9, dtype=torch.float32, device="cuda")
    sp.debug_unpack(d.data_ptr(), b.size, out.data_ptr(), torch.cuda.current_stream().cuda_stream, npol=npol)
    got = out.cpu().numpy()
    assert np.array_equal(got, b.astype(np.float32))
    assert np.array_equal(got.view(np.uint32), b.astype(np.float32).view(np.uint32))


def _front_end(nchan, ntaps, npol, mode, raw, nspec, coeffs=None, window=1):
    torch, sp = _torch(), _sp()
    s = sp.Spec(nchan, ntaps, npol, mode, 1, window)
    if coeffs is not None:
        s.set_coeffs(coeffs)
    d = torch.from_numpy(np.ascontiguousarray(raw).reshape(-1)).cuda()
    out = torch.full((nspec, nchan, 2 * npol), 7e9, dtype=torch.float32, device="cuda")
    s.debug_fir(d.data_ptr(), out.data_ptr(), torch.cuda.current_stream().cuda_stream, nspec=nspec)
    got = out.cpu().numpy()
    info = s.plan_info()
    assert s.spectra_done() == 0 and s.pending() == 0      # the hook leaves the stream state alone
    s.close()
    return got, info


# (nchan, ntaps, npol, the kernel whose front end must be the one that runs)
FRONT_PFB = [(64, 4, 1, "k_engine"), (64, 4, 2, "k_engine"), (1024, 8, 1, "k_engine"), (4096, 5, 2, "k_engine"),
             (1024, 8, 2, "k_fused"), (2048, 8, 2, "k_fused"), (4096, 8, 2, "k_fused"), (8192, 8, 2, "k_fused"),
             (16384, 8, 2, "k_fused"), (32768, 8, 2, "k_fused"), (65536, 8, 2, "k_fused"),
             (8192, 8, 1, "k_passA_pfb16"), (8192, 4, 2, "k_engine pass A"), (131072, 8, 1, "k_fir8"),
             (131072, 8, 2, "k_fused"), (262144, 8, 2, "k_fused"), (524288, 8, 2, "k_fused")]


@pytest.mark.parametrize("nchan,ntaps,npol,kernel", FRONT_PFB)
def test_indexing_bit_exact_with_single_tap_coefficients(nchan, ntaps, npol, kernel):
    """h = delta at tap t0(n) for each branch: the FIR output must equal the selected input sample exactly,
    for every spectrum of a run that spans several producer phases and a ragged tail (SURVEY section 4 tier 2)."""
    nspec = 19 if nchan <= 65536 else 3
    raw = synth.random_bytes(77 + nchan + ntaps, (nspec + ntaps - 1) * nchan, npol)
    rng = np.random.default_rng(nchan)
    t0 = rng.integers(0, ntaps, size=nchan)
    h = np.zeros((ntaps, nchan), dtype=np.float32)
    h[t0, np.arange(nchan)] = 1.0
    got, (n1, n2, desc) = _front_end(nchan, ntaps, npol, PFB, raw, nspec, coeffs=h)
    if kernel is not None:
        assert kernel in desc, desc
    x = raw.reshape(nspec + ntaps - 1, nchan, 2 * npol)
    n = np.arange(nchan)
    for m in range(nspec):
        want = x[m + t0, n].astype(np.float32)
        assert np.array_equal(got[m], want), f"spectrum {m} via {desc}"


FRONT_FFT = [(256, 2, "k_engine"), (4096, 2, "k_engine"), (4096, 1, "k_engine"), (8192, 2, "FrontRawR2"), (16384, 2, "k_fused"),
             (32768, 2, "k_fused"), (65536, 2, "k_fused"), (16384, 1, "k_engine pass A"), (131072, 2, "k_fused"), (262144, 2, "k_fused"), (524288, 2, "k_fused")]


@pytest.mark.parametrize("nchan,npol,kernel", FRONT_FFT)
def test_unpack_and_indexing_bit_exact_direct_fft_front_end(nchan, npol, kernel):
    """Direct-FFT mode, rectangular window: what reaches the first butterfly is the unpacked sample itself.
    Uniform random bytes: every value -128..127 occurs in every byte lane."""
    nspec = 11 if nchan <= 65536 else 3
    raw = synth.random_bytes(5 + nchan, nspec * nchan, npol)
    for lane in range(2 * npol):
        assert np.unique(raw[:, lane]).size == 256
    got, (n1, n2, desc) = _front_end(nchan, 1, npol, FFT, raw, nspec, window=0)
    if kernel is not None:
        assert kernel in desc, desc
    want = raw.reshape(nspec, nchan, 2 * npol).astype(np.float32)
    if "FrontRawR2" in desc:
        # N = 2 L in one launch: the front end hands the L-point transform the first radix-2 layer, [r][e]:
        # r = 0 the sums x[e] + x[e+L] (small integers: exact), r = 1 the differences times W_N^e
        L = nchan // 2
        lo, hi = want[:, :L].astype(np.float64), want[:, L:].astype(np.float64)
        assert np.array_equal(got[:, :L], (lo + hi).astype(np.float32)), desc
        w = np.exp(-2j * np.pi * np.arange(L) / nchan)
        for p in range(npol):
            dz = ((lo[..., 2 * p] - hi[..., 2 * p]) + 1j * (lo[..., 2 * p + 1] - hi[..., 2 * p + 1])) * w
            gz = got[:, L:, 2 * p].astype(np.float64) + 1j * got[:, L:, 2 * p + 1]
            assert np.max(np.abs(gz - dz)) <= 3e-7 * 256 * np.sqrt(2), desc
        return
    assert np.array_equal(got, want), desc
    assert np.array_equal(got.view(np.uint32), want.view(np.uint32))


@pytest.mark.parametrize("nchan,npol", [(2048, 1), (2048, 2), (32768, 2), (131072, 2)])
def test_fir_stage_against_oracle_fir(nchan, npol):
    import oracle
    N, T, nspec = nchan, 8, 10 if nchan <= 32768 else 2
    raw = synth.random_bytes(5, (nspec + T - 1) * N, npol)
    h = synth.random_coeffs(6, T * N)
    got, _ = _front_end(N, T, npol, PFB, raw, nspec, coeffs=h)
    got = got.astype(np.float64)
    x = raw.reshape((nspec + T - 1) * N, npol, 2).astype(np.float64)
    for m in (0, nspec // 2, nspec - 1):
        for p in range(npol):
            seg = x[m * N:(m + T) * N, p]
            y = oracle.fir(h, seg[:, 0] + 1j * seg[:, 1], N, T)
            g = got[m, :, 2 * p] + 1j * got[m, :, 2 * p + 1]
            assert np.linalg.norm(g - y) / np.linalg.norm(y) < 5e-7


# ---------------------------------------------------------------- parity across sizes / modes

SIZES = [16, 32, 64, 128, 256, 512, 1024, 2048, 4096, 8192, 16384, 32768, 65536]


@pytest.mark.parametrize("npol", [2, 1])
@pytest.mark.parametrize("mode", [PFB, FFT])
@pytest.mark.parametrize("nchan", SIZES)
def test_parity_random_bytes_all_kernels(nchan, mode, npol):
    """Full-range random bytes (including -128), arbitrary coefficients, nacc that does not divide
    the spectra count (ragged tail left in progress), three calls of unequal size."""
    T = 5 if mode == PFB else 1
    M = 3
    nblk = 2 * M + (T - 1) + 2
    raw = synth.random_bytes(nchan * 7 + mode * 3 + npol, nblk * nchan, npol)
    h = synth.random_coeffs(nchan + 1, nchan * T)
    splits = [nchan * 2, nchan * (nblk - 5), nchan * 3]
    g, gd = gpu_run(raw, nchan, T, npol, mode, M, coeffs=h, splits=splits)
    r, rd = oracle_run(raw, nchan, T, npol, mode, M, coeffs=h)
    assert gd == rd == nblk - (T - 1)
    assert len(g) == len(r) == 2
    for a, b in zip(g, r):
        compare(a, b, f"N={nchan} mode={mode} P={npol}")
        check_stokes_invariants(a)


FUSED_SIZES = [1024, 2048, 4096, 8192, 16384, 32768, 65536]


@pytest.mark.parametrize("mode", [PFB, FFT])
@pytest.mark.parametrize("nchan", FUSED_SIZES)
def test_parity_fused_persistent_kernel_small_streams(nchan, mode):
    """The persistent four-step kernel (dual-pol, 8 taps / rectangular direct FFT): full-range random
    bytes, arbitrary PFB coefficients, a ragged last group, windows that straddle three unequal calls."""
    T = 8 if mode == PFB else 1
    M = 3
    nblk = 2 * M + (T - 1) + 2
    raw = synth.random_bytes(nchan * 5 + mode, nblk * nchan, 2)
    h = synth.random_coeffs(nchan + 2, nchan * T) if mode == PFB else None
    splits = [nchan * 2, nchan * (nblk - 5), nchan * 3]
    g, gd = gpu_run(raw, nchan, T, 2, mode, M, coeffs=h, window=(1 if mode == PFB else 0), splits=splits)
    r, rd = oracle_run(raw, nchan, T, 2, mode, M, coeffs=h, window=(1 if mode == PFB else 0))
    assert gd == rd == nblk - (T - 1)
    assert len(g) == len(r) == 2
    for a, b in zip(g, r):
        compare(a, b, f"fused N={nchan} mode={mode}")
        check_stokes_invariants(a)


@pytest.mark.parametrize("nchan,mode,nspec,M", [(1024, PFB, 5200, 700), (2048, PFB, 2900, 1000),
                                                (8192, PFB, 700, 97), (8192, FFT, 700, 256),
                                                (32768, FFT, 200, 64), (65536, PFB, 130, 50)])
def test_parity_fused_kernel_ring_wraps(nchan, mode, nspec, M):
    """Streams longer than the L2-resident Z ring: every ring slot is reused, producers wait for
    consumers and back; several accumulation windows per call and a partial one left at the end."""
    T = 8 if mode == PFB else 1
    nblk = nspec + T - 1
    raw = synth.dual_pol_stream(400 + nchan // 1024 + mode, nblk * nchan, [synth.F_CFG1])
    w = 1 if mode == PFB else 0
    g, gd = gpu_run(raw, nchan, T, 2, mode, M, window=w, splits=[nchan * (nblk - 40), nchan * 40], ring=16)
    r, rd = oracle_run(raw, nchan, T, 2, mode, M, window=w)
    assert gd == rd == nspec
    assert len(g) == len(r) == nspec // M
    for a, b in zip(g, r):
        compare(a, b, f"fused ring N={nchan} mode={mode}")


@pytest.mark.parametrize("nchan,mode,nspec,M", [(131072, PFB, 61, 25), (131072, FFT, 50, 16), (262144, PFB, 37, 11),
                                                (262144, FFT, 30, 30), (524288, PFB, 21, 16), (524288, FFT, 19, 6)])
def test_parity_fused_kernel_largest_sizes_ring_wraps(nchan, mode, nspec, M):
    """N >= 131072: the persistent kernel with N1 = 32, 64, 128 column transforms (two-stage, in place in shared
    memory) and 4096-point rows; more spectra than its small L2-resident ring holds, two calls, ragged last group."""
    T = 8 if mode == PFB else 1
    nblk = nspec + T - 1
    raw = synth.dual_pol_stream(500 + nchan // 65536 + mode, nblk * nchan, [synth.F_CFG1])
    w = 1 if mode == PFB else 0
    g, gd = gpu_run(raw, nchan, T, 2, mode, M, window=w, splits=[nchan * (nblk - 9), nchan * 9], ring=16)
    r, rd = oracle_run(raw, nchan, T, 2, mode, M, window=w)
    assert gd == rd == nspec
    assert len(g) == len(r) == nspec // M
    for a, b in zip(g, r):
        compare(a, b, f"fused large N={nchan} mode={mode}")
        check_stokes_invariants(a)


def test_two_handles_on_two_streams_share_the_gpu():
    """Two persistent-kernel handles fed alternately on two CUDA streams: the second launch can only become
    resident as the first one drains (both size their grid to the whole GPU); results must not depend on it."""
    torch, sp = _torch(), _sp()
    cfgs = [(8192, PFB, 8, 40), (32768, FFT, 1, 16)]
    raws = [synth.dual_pol_stream(900 + i, (3 * M + T - 1) * N, [synth.F_CFG1]) for i, (N, mode, T, M) in enumerate(cfgs)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    specs, devs, outs = [], [], [[], []]
    for (N, mode, T, M), raw in zip(cfgs, raws):
        specs.append(sp.Spec(N, T, 2, mode, M, 1 if mode == PFB else 0))
        devs.append(torch.from_numpy(raw.reshape(-1)).cuda())
    torch.cuda.synchronize()
    for part in range(3):   # three calls per handle, interleaved
        for i, ((N, mode, T, M), raw) in enumerate(zip(cfgs, raws)):
            nblk = raw.shape[0] // N
            lo = part * nblk // 3
            hi = (part + 1) * nblk // 3
            specs[i].process(devs[i].data_ptr() + lo * N * 4, (hi - lo) * N, streams[i].cuda_stream)
    for i in range(2):
        while specs[i].pending():
            outs[i].append(specs[i].read_accum_host(streams[i].cuda_stream))
        specs[i].close()
    for i, ((N, mode, T, M), raw) in enumerate(zip(cfgs, raws)):
        r, _ = oracle_run(raw, N, T, 2, mode, M, window=(1 if mode == PFB else 0))
        assert len(outs[i]) == len(r) == 3
        for a, b in zip(outs[i], r):
            compare(a, b, f"two handles N={N}")


@pytest.mark.parametrize("nchan", [131072, 262144, 524288])
def test_parity_largest_channel_counts(nchan):
    T, M = 8, 2
    raw = synth.dual_pol_stream(99, (M + T - 1) * nchan, [synth.F_CFG1])
    g, _ = gpu_run(raw, nchan, T, 2, PFB, M)
    r, _ = oracle_run(raw, nchan, T, 2, PFB, M)
    assert len(g) == len(r) == 1
    compare(g[0], r[0], f"N={nchan}")
    g, _ = gpu_run(raw[: 2 * nchan], nchan, 1, 2, FFT, M, window=0)
    r, _ = oracle_run(raw[: 2 * nchan], nchan, 1, 2, FFT, M, window=0)
    compare(g[0], r[0], f"N={nchan} fft")


def test_split_invariance_many_small_calls():
    """A16: outputs depend only on the concatenated stream: one block per call vs one call."""
    N, T, M = 1024, 8, 4
    raw = synth.dual_pol_stream(3, 40 * N, [synth.F_CFG1])
    a, _ = gpu_run(raw, N, T, 2, PFB, M)
    b, _ = gpu_run(raw, N, T, 2, PFB, M, splits=[N] * 40)
    r, _ = oracle_run(raw, N, T, 2, PFB, M)
    assert len(a) == len(b) == len(r) == 8
    for x, y, z in zip(a, b, r):
        compare(x, z)
        compare(y, z)


@pytest.mark.parametrize("window", [0, 1])
def test_parity_direct_fft_8192_single_launch(window):
    """N = 8192 direct FFT: one k_engine launch, every spectrum as two 4096-point transforms of the first radix-2
    layer (FrontRawR2); rectangular and Hann windows, windows that straddle ragged runs and three calls."""
    N, M, nspec = 8192, 29, 133
    raw = synth.dual_pol_stream(81, nspec * N, [synth.F_CFG1])
    g, gd = gpu_run(raw, N, 1, 2, FFT, M, window=window, splits=[N * 100, N * 1, N * 32])
    r, rd = oracle_run(raw, N, 1, 2, FFT, M, window=window)
    assert gd == rd == nspec and len(g) == len(r) == 4
    for a, b in zip(g, r):
        compare(a, b, f"N=8192 single launch window={window}")
        check_stokes_invariants(a)


def test_hann_window_fft_mode_and_default_coefficients():
    import oracle
    sp = _sp()
    N = 4096
    raw = synth.dual_pol_stream(11, 8 * N, [synth.F_CFG1])
    g, _ = gpu_run(raw, N, 1, 2, FFT, 8, window=1)
    r, _ = oracle_run(raw, N, 1, 2, FFT, 8, window=1)
    compare(g[0], r[0])
    # A20: the library's own default coefficients agree with the oracle's within 1 ulp
    for mode, T in ((PFB, 8), (FFT, 1)):
        s = sp.Spec(N, T, 2, mode, 1, 1)
        mine = s.get_coeffs()
        s.close()
        ref = oracle.default_coeffs(N, T, mode, 1)
        assert np.all(np.abs(mine - ref) <= np.spacing(np.abs(ref).astype(np.float32)))


# ---------------------------------------------------------------- tap counts at the ends of the accepted range

@pytest.mark.parametrize("nchan", [1024, 16384])
@pytest.mark.parametrize("ntaps", [1, 2, 16, 64])
def test_parity_tap_counts(nchan, ntaps):
    """spec_create accepts 1..64 taps: T=1 PFB (a per-branch gain), T=16 and T=64 (the history bookkeeping
    keeps T-1 blocks and the generic FIR loop runs T times)."""
    M = 3
    nblk = 2 * M + (ntaps - 1) + 1
    raw = synth.random_bytes(nchan + ntaps, nblk * nchan, 2)
    h = synth.random_coeffs(ntaps * 3 + 1, nchan * ntaps)
    splits = [nchan * 1, nchan * (nblk - 3), nchan * 2]
    g, gd = gpu_run(raw, nchan, ntaps, 2, PFB, M, coeffs=h, splits=splits)
    r, rd = oracle_run(raw, nchan, ntaps, 2, PFB, M, coeffs=h)
    assert gd == rd == nblk - (ntaps - 1)
    assert len(g) == len(r) == 2
    for a, b in zip(g, r):
        compare(a, b, f"N={nchan} T={ntaps}")


# ---------------------------------------------------------------- back-to-back launches, no sync in between

@pytest.mark.parametrize("mode", [PFB, FFT])
@pytest.mark.parametrize("nchan", FUSED_SIZES)
def test_back_to_back_calls_without_sync(nchan, mode):
    """Consecutive launches of the persistent kernel overlap (programmatic dependent launch) and hand the filter
    history from one to the next inside the kernels: six calls of 7..12 blocks queued with no read and no
    synchronisation in between, from an idle GPU, five times over; results must match the oracle every time."""
    torch, sp = _torch(), _sp()
    T = 8 if mode == PFB else 1
    M = 11
    mult = (1 << 18) // (7 * nchan) + 1      # every call above the small-call threshold: six persistent launches
    sizes = [9 * mult, 7 * mult, 12 * mult, 8 * mult, 10 * mult, 7 * mult]
    M = 11 * mult
    nblk = sum(sizes)
    raw = synth.dual_pol_stream(700 + nchan // 1024 + mode, nblk * nchan, [synth.F_CFG1])
    r, rd = oracle_run(raw, nchan, T, 2, mode, M, window=(1 if mode == PFB else 0))
    d = torch.from_numpy(raw.reshape(-1)).cuda()
    st = torch.cuda.current_stream().cuda_stream
    s = sp.Spec(nchan, T, 2, mode, M, 1 if mode == PFB else 0)
    s.set_ring(16)
    for rep in range(5):
        torch.cuda.synchronize()
        pos = 0
        for n in sizes:
            s.process(d.data_ptr() + pos * nchan * 4, n * nchan, st)
            pos += n
        assert s.spectra_done() == rd
        outs = []
        while s.pending():
            outs.append(s.read_accum_host(st))
        assert len(outs) == len(r)
        for a, b in zip(outs, r):
            compare(a, b, f"back-to-back N={nchan} mode={mode} rep={rep}")
        s.reset()
    s.close()


# ---------------------------------------------------------------- configs[4]: the sweep's accumulation lengths

SWEEP_LOG2 = 26          # samples per point here; configs[4] runs 2^31 (bench.py --sweep), same M/N ratio per sample
SWEEP_POINTS = [(n, m) for m in (FFT, PFB) for n in (1 << k for k in range(10, 20))]


@pytest.fixture(scope="module")
def sweep_refs():
    """One 2^26-sample config-1 stream and the oracle's accumulation for every sweep point: nacc = 2^26/N
    (minus 7 for the PFB), one complete window each, computed in parallel processes."""
    import os
    ns = 1 << SWEEP_LOG2
    path, raw = make_stream_file(synth.SEED_BASE + 4, ns)
    jobs = []
    for n, m in SWEEP_POINTS:
        T = 8 if m == PFB else 1
        jobs.append((n, T, 2, m, ns // n - (T - 1), 1 if m == PFB else 0))
    res = oracle_many(path, ns, jobs)
    yield raw, {pt: r for pt, r in zip(SWEEP_POINTS, res)}
    del raw
    os.unlink(path)


@pytest.mark.parametrize("nchan,mode", SWEEP_POINTS)
def test_sweep_accumulation_lengths(sweep_refs, nchan, mode):
    """configs[4] at its real accumulation lengths per sample (M = 65536 at N=1024 ... 128 at N=524288 over 2^26
    samples), fed in 64 MiB calls like bench.py does; every other point goes through spec_stream_host."""
    torch, sp = _torch(), _sp()
    raw, refs = sweep_refs
    outs_ref, done_ref = refs[(nchan, mode)]
    ns = 1 << SWEEP_LOG2
    T = 8 if mode == PFB else 1
    M = ns // nchan - (T - 1)
    assert len(outs_ref) == 1 and done_ref == M
    streamed = (SWEEP_POINTS.index((nchan, mode)) % 2 == 1)
    st = torch.cuda.current_stream().cuda_stream
    s = sp.Spec(nchan, T, 2, mode, M, 1 if mode == PFB else 0)
    chunk = 1 << 24
    if streamed:
        hp = torch.from_numpy(np.asarray(raw).reshape(-1)).pin_memory()
        assert s.stream_host(hp.data_ptr(), ns, chunk, st) == 1
    else:
        d = torch.from_numpy(np.asarray(raw).reshape(-1)).cuda()
        done = 0
        for c in range(ns // chunk):
            done += s.process(d.data_ptr() + c * chunk * 4, chunk, st)
        assert done == 1
    got = s.read_accum_host(st)
    assert s.spectra_done() == M
    s.close()
    w = compare(got, outs_ref[0], f"sweep N={nchan} mode={mode} M={M} streamed={streamed}")
    check_stokes_invariants(got)
    assert w["rel_l2"] < 3e-5      # far inside the 1e-4 tolerance: no drift from the accumulation length


def test_sweep_longest_accumulation_2e21_spectra(sweep_refs):
    """SURVEY 8(c) A18 / configs[4] at N=1024 direct FFT: M = 2^21 spectra, 2^31 samples.  The device-resident
    2^26-sample buffer is fed 32 times (direct-FFT mode has no memory between blocks, so the accumulation is
    exactly 32 times the oracle's sum over the 2^16 spectra of the buffer, computed in fp64)."""
    torch, sp = _torch(), _sp()
    raw, refs = sweep_refs
    outs_ref, _ = refs[(1024, FFT)]
    N, M, reps = 1024, 1 << 21, 32
    st = torch.cuda.current_stream().cuda_stream
    d = torch.from_numpy(np.asarray(raw).reshape(-1)).cuda()
    s = sp.Spec(N, 1, 2, FFT, M, 0)
    chunk = 1 << 24
    done = 0
    for rep in range(reps):
        for c in range((1 << SWEEP_LOG2) // chunk):
            done += s.process(d.data_ptr() + c * chunk * 4, chunk, st)
    assert done == 1 and s.spectra_done() == M
    got = s.read_accum_host(st)
    s.close()
    w = compare(got, reps * np.asarray(outs_ref[0]), "N=1024 FFT M=2^21")
    assert w["rel_l2"] < 3e-5


# ---------------------------------------------------------------- NEXT-2: first DFT factor on the tensor cores

@pytest.mark.parametrize("nchan", [16384, 32768])
@pytest.mark.parametrize("stream", ["random_bytes", "config1"])
def test_tensor_core_first_stage_parity(nchan, stream):
    """spec_set_option(SPEC_OPT_TENSOR_CORE_STAGE): the 16-point column DFT of the direct-FFT plans as a tcgen05.mma
    contraction (fp16 samples, exact; DFT matrix split into two fp16 terms; fp32 accumulation in tensor memory).
    Same tolerances as every other path (north_star: "only if the stated tolerance still holds"); full-range bytes
    exercise -128 and the largest sums, the config-1 stream a ring that wraps."""
    torch, sp = _torch(), _sp()
    M = 37
    nspec = 3 * M + 5 if stream == "config1" else M + 3
    raw = (synth.dual_pol_stream(1500 + nchan // 1024, nspec * nchan, [synth.F_CFG1]) if stream == "config1"
           else synth.random_bytes(1600 + nchan // 1024, nspec * nchan, 2))
    r, rd = oracle_run(raw, nchan, 1, 2, FFT, M, window=0)
    d = torch.from_numpy(raw.reshape(-1)).cuda()
    st = torch.cuda.current_stream().cuda_stream
    errs = {}
    for tc in (0, 1):
        s = sp.Spec(nchan, 1, 2, FFT, M, 0)
        s.set_option(sp.OPT_TENSOR_CORE_STAGE, tc)
        s.process(d.data_ptr(), (nspec - 7) * nchan, st)
        s.process(d.data_ptr() + (nspec - 7) * nchan * 4, 7 * nchan, st)
        assert s.spectra_done() == rd
        outs = []
        while s.pending():
            outs.append(s.read_accum_host(st))
        s.close()
        assert len(outs) == len(r)
        worst = 0.0
        for a, b in zip(outs, r):
            worst = max(worst, compare(a, b, f"tc={tc} N={nchan} {stream}")["rel_l2"])
            check_stokes_invariants(a)
        errs[tc] = worst
    print(f"N={nchan} {stream}: rel L2 fp32 stage {errs[0]:.2e}, tensor-core stage {errs[1]:.2e}")
    assert errs[1] < 2e-5


def test_tensor_core_option_rejected_where_the_plan_has_no_such_stage():
    sp = _sp()
    for args in ((32768, 8, 2, PFB, 4, 1), (4096, 1, 2, FFT, 4, 0), (8192, 1, 2, FFT, 4, 0), (65536, 1, 2, FFT, 4, 0),
                 (16384, 1, 1, FFT, 4, 0)):
        s = sp.Spec(*args)
        with pytest.raises(sp.SpecError) as e:
            s.set_option(sp.OPT_TENSOR_CORE_STAGE, 1)
        assert e.value.code == sp.ERR_STATE
        s.set_option(sp.OPT_TENSOR_CORE_STAGE, 0)
        s.close()


# ---------------------------------------------------------------- NEXT-4: packet-sized calls replayed as a CUDA graph

@pytest.mark.parametrize("nchan,mode,ntaps", [(1024, PFB, 8), (256, PFB, 4), (8192, FFT, 1)])
def test_cuda_graph_replay_of_packet_sized_calls(nchan, mode, ntaps):
    """A periodic segment of 18 small spec_process calls (8 blocks each) and its read-outs is captured once and
    replayed on fresh input; the filter history and the accumulation windows carry on across replays on the device.
    The host then sums the read-outs in double precision (the CPU thread)."""
    torch, sp = _torch(), _sp()
    T = ntaps if mode == PFB else 1
    M, bpc, ncalls, nrep = 16, 8, 18, 4
    seg_blocks = bpc * ncalls                      # 144 spectra per segment = 9 windows = the ring's period
    raw = synth.dual_pol_stream(1700 + nchan, ((T - 1) + nrep * seg_blocks) * nchan, [synth.F_CFG1])
    w = 1 if mode == PFB else 0
    r, rd = oracle_run(raw, nchan, T, 2, mode, M, window=w)
    assert len(r) == nrep * 9
    s = sp.Spec(nchan, T, 2, mode, M, w)
    st0 = torch.cuda.current_stream().cuda_stream
    d_all = torch.from_numpy(raw.reshape(-1)).cuda()
    if T > 1:
        s.process(d_all.data_ptr(), (T - 1) * nchan, st0)          # fill the history outside the graph
    seg_bytes = seg_blocks * nchan * 4
    d_seg = torch.empty(seg_bytes, dtype=torch.int8, device="cuda")
    d_out = torch.zeros((9, 4, nchan), dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        st = torch.cuda.current_stream().cuda_stream
        s.capture_begin()
        got = 0
        for c in range(ncalls):
            s.process(d_seg.data_ptr() + c * bpc * nchan * 4, bpc * nchan, st)
            if c % 6 == 5:
                got += s.read_accum_batch_device(d_out.data_ptr() + got * 4 * nchan * 4, 8, st)
        assert got == 9
        s.capture_end()
    outs = []
    hist = (T - 1) * nchan * 4
    for rep in range(nrep):
        d_seg.copy_(d_all[hist + rep * seg_bytes: hist + (rep + 1) * seg_bytes])
        g.replay()
        outs += list(d_out.cpu().numpy())
    s.replayed(nrep - 1)
    assert s.spectra_done() == rd and s.pending() == 0
    s.close()
    total = np.zeros((4, nchan), dtype=np.float64)
    for a, b in zip(outs, r):
        compare(a, b, f"graph replay N={nchan}")
        sp.accumulate_host(total, np.ascontiguousarray(a))
    compare(total, np.sum(np.asarray(r), axis=0), "host-side long accumulation")


def test_cuda_graph_capture_rejects_a_segment_that_is_not_periodic():
    torch, sp = _torch(), _sp()
    N = 1024
    s = sp.Spec(N, 8, 2, PFB, 16)
    d = torch.zeros(64 * N * 4, dtype=torch.int8, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    s.process(d.data_ptr(), 7 * N, st)
    torch.cuda.synchronize()
    s.capture_begin()                     # (no stream capture needed to exercise the bookkeeping)
    for c in range(5):                    # 5 calls: the history buffers and ring parities do not line up again
        s.process(d.data_ptr(), 8 * N, st)
    while s.pending():
        s.read_accum_host(st)
    with pytest.raises(sp.SpecError) as e:
        s.capture_end()
    assert e.value.code == sp.ERR_STATE
    s.close()


# ---------------------------------------------------------------- NEXT-3: eight-sub-band modes

@pytest.mark.parametrize("nchan,mode,ntaps,nsub,npol", [(4096, PFB, 8, 8, 2), (16384, PFB, 8, 8, 2), (65536, PFB, 8, 8, 2),
                                                        (4096, FFT, 1, 8, 2), (8192, FFT, 1, 8, 2), (1024, PFB, 4, 3, 1)])
def test_parity_sub_band_modes(nchan, mode, ntaps, nsub, npol):
    """eight sub-bands x two polarisations = 16 transforms per spectrum set, channel counts of
    Table 1's third block; the input interleaves the sub-bands per time sample (reading R26).  Different data in
    every sub-band (each gets its own tone), two calls, windows that straddle them."""
    import oracle
    torch, sp = _torch(), _sp()
    T = ntaps if mode == PFB else 1
    M = 5
    nblk = 2 * M + (T - 1) + 3
    ns = nblk * nchan
    rng = np.random.default_rng(nchan + nsub)
    raw = rng.integers(-40, 41, size=(ns, nsub, 2 * npol)).astype(np.float64)
    j = np.arange(ns)
    for s in range(nsub):   # a tone of its own per sub-band, in polarisation 0
        z = 30.0 * np.exp(2j * np.pi * ((37 + 11 * s) % nchan) * j / nchan)
        raw[:, s, 0] += z.real
        raw[:, s, 1] += z.imag
    raw = np.clip(np.rint(raw), -128, 127).astype(np.int8)
    w = 1 if mode == PFB else 0
    o = oracle.OracleSub(nsub, nchan, T, npol, mode, M, w)
    o.process(raw)
    ref = []
    while o.pending():
        ref.append(o.read_accum())
    rd = o.spectra_done()
    o.close()
    s_ = sp.Spec(nchan, T, npol, mode, M, w, nsub=nsub)
    n1, n2, desc = s_.plan_info()
    assert f"{nsub} sub-bands" in desc
    d = torch.from_numpy(raw.reshape(-1)).cuda()
    st = torch.cuda.current_stream().cuda_stream
    bps = nsub * 2 * npol
    first = (nblk - 4) * nchan
    got = []
    done = s_.process(d.data_ptr(), first, st)
    done += s_.process(d.data_ptr() + first * bps, ns - first, st)
    assert done == len(ref) == 2 and s_.spectra_done() == rd
    while s_.pending():
        got.append(s_.read_accum_host(st))
    s_.close()
    for a, b in zip(got, ref):
        assert a.shape == b.shape == (nsub, 4 if npol == 2 else 1, nchan)
        for s in range(nsub):
            compare(a[s], b[s], f"sub-band {s} of {nsub}, N={nchan} mode={mode}")
            assert np.argmax(a[s][0]) == (37 + 11 * s) % nchan


def test_sub_band_stream_host_and_batch_read():
    torch, sp = _torch(), _sp()
    import oracle
    N, T, M, nsub = 4096, 8, 4, 8
    nblk = 3 * M + T - 1
    rng = np.random.default_rng(99)
    raw = rng.integers(-128, 128, size=(nblk * N, nsub, 4), dtype=np.int8)
    o = oracle.OracleSub(nsub, N, T, 2, oracle.MODE_PFB, M)
    o.process(raw)
    ref = [o.read_accum() for _ in range(3)]
    o.close()
    hp = torch.from_numpy(raw.reshape(-1)).pin_memory()
    st = torch.cuda.current_stream().cuda_stream
    s = sp.Spec(N, T, 2, PFB, M, nsub=nsub)
    assert s.stream_host(hp.data_ptr(), nblk * N, 5 * N, st) == 3
    out = torch.zeros((3, nsub, 4, N), dtype=torch.float32, device="cuda")
    assert s.read_accum_batch_device(out.data_ptr(), 8, st) == 3
    got = out.cpu().numpy()
    s.close()
    for c in range(3):
        for k in range(nsub):
            compare(got[c, k], ref[c][k], f"sub-band batch read {c}/{k}")


# ---------------------------------------------------------------- BASELINE.json configs

def _run_config(cfg, ring=None):
    c = synth.CONFIGS[cfg]
    raw = synth.config_stream(cfg)
    mode = PFB if c["mode"] == "pfb" else FFT
    window = 1 if mode == PFB else 0
    per = c["nsamples"] // c["calls"]
    g, gd = gpu_run(raw, c["nchan"], c["ntaps"], c["npol"], mode, c["nacc"], window=window,
                    splits=[per] * c["calls"], ring=ring)
    r, rd = oracle_run(raw, c["nchan"], c["ntaps"], c["npol"], mode, c["nacc"], window=window)
    assert gd == rd
    assert len(g) == len(r)
    worst = {}
    for a, b in zip(g, r):
        worst = compare(a, b, c["name"])
        check_stokes_invariants(a)
    return g, r, worst


def test_config0_single_pol_pfb_1k():
    g, r, _ = _run_config(0)
    assert len(g) == 1 and g[0].shape == (1, 1024)
    # SURVEY 8c expected values: tone at channel 100, half-channel tone split over 300/301
    assert np.argmax(g[0][0]) == 100
    assert abs(g[0][0][300] / g[0][0][301] - 1) < 0.1


def test_config2_direct_fft_4k():
    g, r, _ = _run_config(2)
    assert len(g) == 1 and g[0].shape == (4, 4096)
    # A11: correlated generator, phase of sum(XY*) -> -pi/5
    ph = np.angle(np.sum(g[0][2].astype(np.float64)) + 1j * np.sum(g[0][3].astype(np.float64)))
    assert abs(ph + np.pi / 5) < 0.02


def test_config3_pfb_512k_four_step():
    g, r, _ = _run_config(3)
    assert len(g) == 1 and g[0].shape == (4, 524288)
    assert np.argmax(g[0][0]) == 1000


def test_config1_pfb_32k_streamed_64MiB_calls():
    g, r, _ = _run_config(1)
    assert len(g) == 7  # 2041 spectra, M=256: windows straddle the 64 MiB calls
    # the call pattern bench.py times: the four 64 MiB calls queued back to back (overlapping persistent launches,
    # history handed over inside the kernels), no read and no synchronisation in between, ONE batched read-out at the end
    torch, sp = _torch(), _sp()
    c = synth.CONFIGS[1]
    raw = synth.config_stream(1)
    d = torch.from_numpy(raw.reshape(-1)).cuda()
    st = torch.cuda.current_stream().cuda_stream
    s = sp.Spec(c["nchan"], c["ntaps"], 2, PFB, c["nacc"], 1)
    s.set_ring(16)
    out = torch.zeros((16, 4, c["nchan"]), dtype=torch.float32, device="cuda")
    per = c["nsamples"] // c["calls"]
    for rep in range(3):
        torch.cuda.synchronize()
        for k in range(c["calls"]):
            s.process(d.data_ptr() + k * per * 4, per, st)
        assert s.read_accum_batch_device(out.data_ptr(), 16, st) == 7
        got = out[:7].cpu().numpy()
        for a, b in zip(got, r):
            compare(a, b, f"configs[1], bench.py's call pattern, repetition {rep}")
        s.reset()
    s.close()


# ---------------------------------------------------------------- API behaviour on the device

def test_api_errors_and_ring():
    torch, sp = _torch(), _sp()
    N = 256
    s = sp.Spec(N, 4, 2, PFB, 1)
    d = torch.zeros(64 * N * 4, dtype=torch.int8, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    with pytest.raises(sp.SpecError) as e:
        s.process(d.data_ptr(), N + 1, st)
    assert e.value.code == sp.ERR_SIZE
    with pytest.raises(sp.SpecError) as e:
        s.set_coeffs(np.zeros(N * 4 + 1, np.float32))
    assert e.value.code == sp.ERR_SIZE
    assert s.process(d.data_ptr(), 0, st) == 0
    assert s.read_accum_host(st) is None
    assert s.process(d.data_ptr(), 3 * N, st) == 0           # history filling, no spectrum yet
    assert s.spectra_done() == 0
    assert s.process(d.data_ptr(), 8 * N, st) == 8           # M=1: 8 outputs fill the ring
    assert s.pending() == 8
    with pytest.raises(sp.SpecError) as e:
        s.process(d.data_ptr(), N, st)                       # a 9th would overrun
    assert e.value.code == sp.ERR_OVERRUN
    assert s.spectra_done() == 8                             # state unchanged by the failed call
    assert s.read_accum_host(st) is not None
    assert s.process(d.data_ptr(), N, st) == 1
    with pytest.raises(sp.SpecError) as e:
        s.set_ring(16)                                       # only after create/reset
    assert e.value.code == sp.ERR_STATE
    s.reset()
    assert s.pending() == 0 and s.spectra_done() == 0
    s.set_ring(16)
    assert s.process(d.data_ptr(), 19 * N, st) == 16
    s.close()


def test_read_accum_to_device_matches_host():
    torch, sp = _torch(), _sp()
    N = 2048
    raw = synth.dual_pol_stream(5, 12 * N, [synth.F_CFG1])
    d = torch.from_numpy(raw.reshape(-1)).cuda()
    st = torch.cuda.current_stream().cuda_stream
    outs = []
    for to_dev in (True, False):
        s = sp.Spec(N, 8, 2, PFB, 5)
        assert s.process(d.data_ptr(), 12 * N, st) == 1
        if to_dev:
            o = torch.empty((4, N), dtype=torch.float32, device="cuda")
            assert s.read_accum_device(o.data_ptr(), st) == 1
            outs.append(o.cpu().numpy())
        else:
            outs.append(s.read_accum_host(st))
        s.close()
    r, _ = oracle_run(raw, N, 8, 2, PFB, 5)
    compare(outs[0], r[0])
    compare(outs[1], r[0])


def test_read_accum_batch_matches_oracle_across_ring_wrap():
    """spec_read_accum_batch: several accumulations per launch, oldest first, slots wrapping around the ring."""
    torch, sp = _torch(), _sp()
    N, T, M = 2048, 8, 3
    nblk = 11 * M + T - 1
    raw = synth.dual_pol_stream(33, nblk * N, [synth.F_CFG1])
    d = torch.from_numpy(raw.reshape(-1)).cuda()
    st = torch.cuda.current_stream().cuda_stream
    s = sp.Spec(N, T, 2, PFB, M)           # default ring: 8 slots
    o = torch.zeros((8, 4, N), dtype=torch.float32, device="cuda")
    got = []
    first = (5 * M + T - 1) * N
    assert s.process(d.data_ptr(), first, st) == 5
    assert s.read_accum_batch_device(o.data_ptr(), 4, st) == 4        # max_count honoured
    got += list(o[:4].cpu().numpy())
    assert s.pending() == 1
    assert s.process(d.data_ptr() + first * 4, nblk * N - first, st) == 6   # slots 5,6,7,0,1,2: wraps
    assert s.read_accum_batch_device(o.data_ptr(), 8, st) == 7
    got += list(o[:7].cpu().numpy())
    assert s.read_accum_batch_device(o.data_ptr(), 8, st) == 0
    s.close()
    r, _ = oracle_run(raw, N, T, 2, PFB, M)
    assert len(r) == 11
    for a, b in zip(got, r):
        compare(a, b)


def test_stream_host_double_buffered_matches_oracle():
    """north_star item (d): pinned host memory, two device buffers, side-stream copies."""
    torch, sp = _torch(), _sp()
    N, T, M = 4096, 8, 16
    nblk = 3 * M + T - 1 + 5
    raw = synth.dual_pol_stream(21, nblk * N, [synth.F_CFG1])
    hp = torch.from_numpy(raw.reshape(-1)).pin_memory()
    st = torch.cuda.current_stream().cuda_stream
    s = sp.Spec(N, T, 2, PFB, M)
    done = s.stream_host(hp.data_ptr(), nblk * N, 7 * N, st)   # ragged last chunk
    assert done == 3
    g = [s.read_accum_host(st) for _ in range(3)]
    s.close()
    r, _ = oracle_run(raw, N, T, 2, PFB, M)
    for a, b in zip(g, r):
        compare(a, b)


def test_long_accumulation_two_level_sum():
    """A18: many spectra per window: per-CTA register sums, then atomics; error stays far below 1e-4."""
    N, M = 1024, 8192
    raw = synth.dual_pol_stream(8, M * N, [synth.F_CFG1])
    g, _ = gpu_run(raw, N, 1, 2, FFT, M, window=0)
    r, _ = oracle_run(raw, N, 1, 2, FFT, M, window=0)
    w = compare(g[0], r[0])
    assert w["rel_l2"] < 2e-5


def test_fp32_peak_probe_runs():
    sp = _sp()
    tf = sp.measure_fp32_peak(0)
    assert 20.0 < tf < 100.0

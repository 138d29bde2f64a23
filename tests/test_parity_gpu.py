"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle on the same seeded
inputs.  Bit-exact for the unpack and indexing stages, BASELINE.json north_star tolerances for the
accumulated spectra (tests/_harness.py)."""
import numpy as np
import pytest

from _harness import check_stokes_invariants, compare, gpu_run, oracle_run
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

def test_unpack_bit_exact_all_values_all_lanes():
    torch, sp = _torch(), _sp()
    # every byte value in every byte lane of a 32-bit word, plus a ragged tail (1027 bytes)
    vals = np.arange(-128, 128, dtype=np.int8)
    b = np.concatenate([np.roll(vals, k) for k in range(4)] + [vals[:3]]).astype(np.int8)
    d = torch.from_numpy(b).cuda()
    out = torch.full((b.size,), 1e9, dtype=torch.float32, device="cuda")
    sp.debug_unpack(d.data_ptr(), b.size, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    got = out.cpu().numpy()
    assert np.array_equal(got, b.astype(np.float32))
    assert np.array_equal(got.view(np.uint32), b.astype(np.float32).view(np.uint32))


@pytest.mark.parametrize("npol", [1, 2])
@pytest.mark.parametrize("nchan,ntaps", [(64, 4), (1024, 8), (8192, 8)])
def test_indexing_bit_exact_with_single_tap_coefficients(nchan, ntaps, npol):
    """h = delta at tap t0(n) for each branch: the FIR output must equal the selected input
    sample exactly (SURVEY section 4 tier 2)."""
    torch, sp = _torch(), _sp()
    raw = synth.random_bytes(77 + nchan, ntaps * nchan, npol)
    rng = np.random.default_rng(nchan)
    t0 = rng.integers(0, ntaps, size=nchan)
    h = np.zeros((ntaps, nchan), dtype=np.float32)
    h[t0, np.arange(nchan)] = 1.0
    s = sp.Spec(nchan, ntaps, npol, PFB, 1)
    s.set_coeffs(h)
    d = torch.from_numpy(raw.reshape(-1)).cuda()
    out = torch.zeros((nchan, 2 * npol), dtype=torch.float32, device="cuda")
    s.debug_fir(d.data_ptr(), out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    got = out.cpu().numpy()
    s.close()
    want = raw.reshape(ntaps, nchan, 2 * npol)[t0, np.arange(nchan)].astype(np.float32)
    assert np.array_equal(got, want)


@pytest.mark.parametrize("npol", [1, 2])
def test_fir_stage_against_oracle_fir(npol):
    import oracle
    torch, sp = _torch(), _sp()
    N, T = 2048, 8
    raw = synth.random_bytes(5, T * N, npol)
    h = synth.random_coeffs(6, T * N)
    s = sp.Spec(N, T, npol, PFB, 1)
    s.set_coeffs(h)
    d = torch.from_numpy(raw.reshape(-1)).cuda()
    out = torch.zeros((N, 2 * npol), dtype=torch.float32, device="cuda")
    s.debug_fir(d.data_ptr(), out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    got = out.cpu().numpy().astype(np.float64)
    s.close()
    x = raw.reshape(T * N, npol, 2).astype(np.float64)
    for p in range(npol):
        y = oracle.fir(h, x[:, p, 0] + 1j * x[:, p, 1], N, T)
        g = got[:, 2 * p] + 1j * got[:, 2 * p + 1]
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

"""Shared helpers of the GPU parity tests: run a stream through the CUDA library (via the C ABI)
and through the CPU oracle, and compare with the tolerances BASELINE.json north_star states:
relative L2 <= 1e-4 over each accumulated spectrum (per Stokes plane) and per-channel relative
error <= 1e-3 on channels holding more than 1e-6 of the plane's total power (DESIGN.md reading
R17 for the signed cross-product planes)."""
import numpy as np

import oracle

REL_L2 = 1e-4
REL_CH = 1e-3
CH_FLOOR = 1e-6


def gpu_run(raw, nchan, ntaps, npol, mode, nacc, coeffs=None, window=1, splits=None, ring=None):
    """raw: int8 [nsamples, 2*npol].  splits: list of per-call sample counts (default: one call).
    Returns (list of float32 [S, nchan] outputs, spectra_done)."""
    import torch

    from paper_1411_0436_b200 import spec as sp

    s = sp.Spec(nchan, ntaps, npol, mode, nacc, window)
    try:
        if ring:
            s.set_ring(ring)
        if coeffs is not None:
            s.set_coeffs(coeffs)
        raw = np.ascontiguousarray(raw, dtype=np.int8)
        ns = raw.shape[0]
        d = torch.from_numpy(raw.reshape(-1)).cuda()
        stream = torch.cuda.current_stream().cuda_stream
        outs = []
        pos = 0
        bps = 2 * npol
        for n in (splits or [ns]):
            s.process(d.data_ptr() + pos * bps, n, stream)
            pos += n
            while s.pending():
                outs.append(s.read_accum_host(stream))
        assert pos == ns
        torch.cuda.synchronize()
        return outs, s.spectra_done()
    finally:
        s.close()


def oracle_run(raw, nchan, ntaps, npol, mode, nacc, coeffs=None, window=1):
    o = oracle.Oracle(nchan, ntaps, npol, mode, nacc, window)
    if coeffs is not None:
        o.set_coeffs(coeffs)
    o.process(raw)
    outs = []
    while o.pending():
        outs.append(o.read_accum())
    done = o.spectra_done()
    o.close()
    return outs, done


def compare(gpu, ref, what=""):
    """gpu: float32 [S,N]; ref: float64 [S,N].  Returns dict of worst errors; asserts tolerances."""
    gpu = np.asarray(gpu, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert gpu.shape == ref.shape, (gpu.shape, ref.shape)
    S = ref.shape[0]
    worst = {"rel_l2": 0.0, "rel_ch": 0.0}
    for p in range(S):
        g, r = gpu[p], ref[p]
        nr = np.linalg.norm(r)
        if S == 4 and p >= 2:
            scale = np.sqrt(np.abs(ref[0] * ref[1]))
            nr = max(nr, 1e-3 * np.linalg.norm(scale))
        if nr == 0:
            assert np.all(g == 0), f"{what}: plane {p} should be zero"
            continue
        l2 = np.linalg.norm(g - r) / nr
        worst["rel_l2"] = max(worst["rel_l2"], l2)
        assert l2 <= REL_L2, f"{what}: plane {p} relative L2 {l2:.3e} > {REL_L2}"
        tot = np.sum(np.abs(r))
        sel = np.abs(r) > CH_FLOOR * tot
        den = np.abs(r)
        if S == 4 and p >= 2:
            den = np.maximum(den, 1e-3 * scale)
        if np.any(sel):
            e = np.max(np.abs(g - r)[sel] / den[sel])
            worst["rel_ch"] = max(worst["rel_ch"], e)
            assert e <= REL_CH, f"{what}: plane {p} per-channel relative error {e:.3e} > {REL_CH}"
    return worst


def check_stokes_invariants(out, slack=1e-5):
    """XX, YY >= 0 and Re^2 + Im^2 <= XX*YY (Cauchy-Schwarz)."""
    out = np.asarray(out, dtype=np.float64)
    assert np.all(out[0] >= 0)
    if out.shape[0] == 4:
        assert np.all(out[1] >= 0)
        assert np.all(out[2] ** 2 + out[3] ** 2 <= out[0] * out[1] * (1 + slack) + 1e-30)


# ---------------------------------------------------------------- many oracle runs at once
# The oracle is single-threaded C with one static twiddle table, so independent runs go to separate
# PROCESSES (spawned: the parent may hold a CUDA context).  The stream is shared through a file in /dev/shm.

def _oracle_job(args):
    path, nsamples, nchan, ntaps, npol, mode, nacc, window = args
    raw = np.memmap(path, dtype=np.int8, mode="r", shape=(nsamples, 2 * npol))
    outs, done = oracle_run(raw, nchan, ntaps, npol, mode, nacc, window=window)
    return [np.asarray(o) for o in outs], done


def _synth_job(args):
    seed, start, n = args
    from fractions import Fraction  # noqa: F401
    from paper_1411_0436_b200 import synth
    return synth.dual_pol_stream(seed, n, [synth.F_CFG1], start=start)


def make_stream_file(seed, nsamples, workers=None):
    """The config-1 generator's first `nsamples` dual-pol samples as a file in shared memory (generated in
    parallel: chunks of the stream are independent by construction).  Returns (path, int8 array view)."""
    import concurrent.futures as cf
    import multiprocessing as mp
    import os
    import tempfile
    workers = workers or min(16, os.cpu_count() or 1)
    d = "/dev/shm" if os.path.isdir("/dev/shm") else tempfile.gettempdir()
    path = os.path.join(d, f"spec_stream_{os.getpid()}_{seed}_{nsamples}.i8")
    out = np.memmap(path, dtype=np.int8, mode="w+", shape=(nsamples, 4))
    piece = 1 << 22
    jobs = [(seed, s, min(piece, nsamples - s)) for s in range(0, nsamples, piece)]
    with cf.ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn")) as ex:
        for (sd, s, n), r in zip(jobs, ex.map(_synth_job, jobs)):
            out[s:s + n] = r
    out.flush()
    return path, out


def oracle_many(path, nsamples, jobs, workers=None):
    """jobs: list of (nchan, ntaps, npol, mode, nacc, window) on the first nsamples of the stream file.
    Returns a list of (outputs, spectra_done) in the same order, computed in parallel processes."""
    import concurrent.futures as cf
    import multiprocessing as mp
    import os
    workers = workers or min(len(jobs), os.cpu_count() or 1)
    args = [(path, nsamples) + tuple(j) for j in jobs]
    with cf.ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn")) as ex:
        return list(ex.map(_oracle_job, args))

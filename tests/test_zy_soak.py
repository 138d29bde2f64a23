"""Soak test of the persistent kernels: more than 200 back-to-back launches per handle with random
call sizes, three handles on three streams, a foreign kernel in the middle.  In a file of its own, collected after the
parity tests and before tests/test_zz_no_alloc.py: it is the one test here that exercises scheduling luck (it found two
real hazards this round, profiles/r02_experiments.md rows 26-27), and the suite runs with pytest -x."""
import numpy as np
import pytest

from _harness import compare, oracle_run
from paper_1411_0436_b200 import synth

pytestmark = pytest.mark.gpu

PFB, FFT = 0, 1


def _torch():
    import torch
    return torch


def _sp():
    from paper_1411_0436_b200 import spec as sp
    return sp


def test_soak_random_call_sizes_two_handles_and_a_foreign_kernel():
    """More than 200 back-to-back launches per handle with random call sizes (some shorter than the T-1 = 7
    blocks of history, so both history-carry paths alternate), two handles on two streams, and a foreign kernel
    that takes every SM's shared memory for 50 ms in the middle of it on a third stream."""
    torch, sp = _torch(), _sp()
    cfgs = [(8192, PFB, 8, 397), (32768, FFT, 1, 64), (1024, PFB, 8, 5000)]
    rng = np.random.default_rng(2026)
    ncalls = 220
    plans, raws, specs, devs = [], [], [], []
    for i, (N, mode, T, M) in enumerate(cfgs):
        big = (1 << 19) // N + 25               # calls on both sides of the small-call threshold (2^18 samples)
        sizes = rng.integers(1, big, size=ncalls)
        sizes[rng.integers(0, ncalls, size=40)] = rng.integers(1, 7, size=40)   # plenty of calls below T-1 blocks
        plans.append(sizes)
        raws.append(synth.dual_pol_stream(1200 + i, int(sizes.sum()) * N, [synth.F_CFG1]))
        specs.append(sp.Spec(N, T, 2, mode, M, 1 if mode == PFB else 0))
        specs[-1].set_ring(64)
        devs.append(torch.from_numpy(raws[-1].reshape(-1)).cuda())
    streams = [torch.cuda.Stream() for _ in cfgs]
    hog_stream = torch.cuda.Stream()
    outs = [[] for _ in cfgs]
    pos = [0] * len(cfgs)
    torch.cuda.synchronize()
    for c in range(ncalls):
        for i, (N, mode, T, M) in enumerate(cfgs):
            n = int(plans[i][c])
            specs[i].process(devs[i].data_ptr() + pos[i] * N * 4, n * N, streams[i].cuda_stream)
            pos[i] += n
            if specs[i].pending() > 40:      # drain now and then (the only reads; no other synchronisation)
                while specs[i].pending():
                    outs[i].append(specs[i].read_accum_host(streams[i].cuda_stream))
        if c == ncalls // 2:
            sp.debug_hog(50, 200 * 1024, hog_stream.cuda_stream)
    for i in range(len(cfgs)):
        while specs[i].pending():
            outs[i].append(specs[i].read_accum_host(streams[i].cuda_stream))
        specs[i].close()
    torch.cuda.synchronize()
    for i, (N, mode, T, M) in enumerate(cfgs):
        r, _ = oracle_run(raws[i], N, T, 2, mode, M, window=(1 if mode == PFB else 0))
        assert len(outs[i]) == len(r) and len(r) >= 2
        for a, b in zip(outs[i], r):
            compare(a, b, f"soak N={N}")

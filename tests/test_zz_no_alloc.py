"""spec_oneshot_static: the entry point that allocates nothing (its scratch is a file-scope device array inside the
library) against the existing handle-based path, on the same inputs, with the tolerances of the parity tests
(tests/_harness.py: relative L2 1e-4 per plane, per-channel 1e-3).  Collected last on purpose (file name): the suite
runs with pytest -x.  Passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from _harness import compare
from paper_1411_0436_b200 import synth

pytestmark = pytest.mark.gpu

PFB, FFT = 0, 1


def _existing_path(raw, nchan, ntaps, npol, mode, nspec, coeffs=None):
    """One accumulation of nspec spectra through a spec_create handle."""
    import torch
    from paper_1411_0436_b200 import spec as sp
    s = sp.Spec(nchan, ntaps, npol, mode, nspec, 0 if mode == FFT else 1)
    if coeffs is not None:
        s.set_coeffs(coeffs)
    d = torch.from_numpy(np.ascontiguousarray(raw).reshape(-1)).cuda()
    st = torch.cuda.current_stream().cuda_stream
    assert s.process(d.data_ptr(), raw.shape[0], st) == 1
    out = s.read_accum_host(st)
    s.close()
    return out


def _oneshot(raw, nchan, ntaps, npol, coeffs=None, check_mem=False):
    import torch
    from paper_1411_0436_b200 import spec as sp
    d = torch.from_numpy(np.ascontiguousarray(raw).reshape(-1)).cuda()
    dc = torch.from_numpy(np.ascontiguousarray(coeffs, dtype=np.float32)).cuda() if coeffs is not None else None
    S = 4 if npol == 2 else 1
    out = torch.full((S, nchan), 3e33, dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    free0 = torch.cuda.mem_get_info()[0]
    n = sp.oneshot_static(d.data_ptr(), raw.shape[0], nchan, out.data_ptr(), ntaps=ntaps, npol=npol,
                          d_coeffs_ptr=(dc.data_ptr() if dc is not None else None), stream=st)
    torch.cuda.synchronize()
    if check_mem:   # (not on the first use of a kernel: the driver loads its code lazily, which takes device memory)
        assert torch.cuda.mem_get_info()[0] >= free0    # the call took no device memory
    return out.cpu().numpy(), n


def test_oneshot_static_matches_the_existing_path_on_two_calls_in_a_row():
    """Direct FFT, N = 4096 (the largest the static array holds), dual-pol: two calls in a row on DIFFERENT data (the
    array keeps the first call's sums and tables: the second result must not see them), then the first data again."""
    N, nspec = 4096, 37
    a = synth.dual_pol_stream(2101, nspec * N, [synth.F_CFG1])
    b = synth.random_bytes(2102, nspec * N, 2)
    want_a = _existing_path(a, N, 1, 2, FFT, nspec)
    want_b = _existing_path(b, N, 1, 2, FFT, nspec)
    got_a, n = _oneshot(a, N, 1, 2)
    assert n == nspec
    got_b, _ = _oneshot(b, N, 1, 2, check_mem=True)
    got_a2, _ = _oneshot(a, N, 1, 2, check_mem=True)
    compare(got_a, want_a.astype(np.float64), "one-shot, first call")
    compare(got_b, want_b.astype(np.float64), "one-shot, second call in a row")
    compare(got_a2, want_a.astype(np.float64), "one-shot, third call")
    # nothing of call two leaked into call three (not bit-equal: several CTAs add their partial sums to a channel with
    # fp32 reductions whose order varies from run to run)
    assert np.max(np.abs(got_a2[:2] - got_a[:2]) / got_a[:2]) < 2e-6


def test_oneshot_static_other_shapes_share_the_array():
    """The channel count changes between calls (tables re-uploaded), PFB with device coefficients, single-pol."""
    for (N, T, P, mode) in ((1024, 8, 2, PFB), (256, 1, 1, FFT), (2048, 4, 1, PFB), (1024, 8, 2, PFB), (64, 1, 2, FFT)):
        nspec = 9
        raw = synth.random_bytes(2200 + N + T, (nspec + T - 1) * N, P)
        h = synth.random_coeffs(2300 + N, T * N) if mode == PFB else None
        want = _existing_path(raw, N, T, P, mode, nspec, coeffs=h)
        got, n = _oneshot(raw, N, T, P, coeffs=h)
        assert n == nspec
        compare(got, want.astype(np.float64), f"one-shot N={N} T={T} P={P}")


def test_oneshot_static_rejects_sizes_beyond_the_array():
    import torch
    from paper_1411_0436_b200 import spec as sp
    d = torch.zeros(8192 * 4, dtype=torch.int8, device="cuda")
    out = torch.zeros((4, 8192), dtype=torch.float32, device="cuda")
    with pytest.raises(sp.SpecError) as e:
        sp.oneshot_static(d.data_ptr(), 8192, 8192, out.data_ptr())
    assert e.value.code == sp.ERR_SIZE and "4096" in str(e.value)
    with pytest.raises(sp.SpecError) as e:
        sp.oneshot_static(d.data_ptr(), 1000, 1024, out.data_ptr())          # not a multiple of nchan
    assert e.value.code == sp.ERR_SIZE
    with pytest.raises(sp.SpecError) as e:
        sp.oneshot_static(d.data_ptr(), 4 * 1024, 1024, out.data_ptr(), ntaps=8)   # taps without coefficients
    assert e.value.code == sp.ERR_ARG

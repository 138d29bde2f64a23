#!/usr/bin/env python
"""bench.py — sustained dual-pol bandwidth of the spectrometer hot path on B200.

Metric (BASELINE.json): complex samples/s per polarisation (= per-polarisation bandwidth) in GHz,
PFB mode by default on configs[1]: dual-pol PFB, N=32768, T=8, M=256, fed in 64 MiB calls that carry
the 7*N filter history.  One "step" = a whole number of passes over a 256 MiB device-resident stream
(four 64 MiB calls per pass, larger than the 126 MB L2), as many passes as make a step last about
60 ms, so that the default 20 steps give a timed region of more than a second; every pass goes through
the whole chain unpack -> FIR -> FFT -> Stokes -> accumulate -> read-out.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                  [--nchan N --mode pfb|fft --nacc M]   (another workload, same JSON line)
  python bench.py --sweep [--sweep-log2 31]             (configs[4]: 20 points, resident and streamed)

`value`  : inputs resident in HBM before the timed region.
`e2e`    : the same work through spec_stream_host from PINNED HOST memory (H2D inside the timed
           region, double-buffered on a side stream) plus a device-to-host copy of every completed
           accumulation into pinned host memory (on a third stream, inside the timed region).
`roofline`: dominant kernel's nominal fp32 flops / its time vs the fp32 peak measured in this run
           (spec_measure_fp32_peak).  Where one kernel is the whole chain its time is taken from the timed
           pass itself ((step time - read-out kernels) / launches: the launches overlap there, no event sits
           between them); `frac_event_bracketed` is the same from a second pass with CUDA events around
           every launch.  `roofline_chain` is north_star's whole-chain roofline.
`cpu_baseline`: the CPU oracle (oracle/, fp64) timed on a bounded sample, on one core and on all cores
           (independent stretches of the stream in separate processes).
`--impl reference` times the oracle alone (the reference arm of this tier).
Multi-GPU: the path shards over independent streams (one beam per GPU): every rank
runs its own stream, no data-path collective, "scaling": "weak".
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

CHUNK_BYTES = 64 << 20      # 64 MiB calls (configs[1])
CALLS_PER_PASS = 4          # one pass = the 256 MiB device-resident stream (four 64 MiB calls)
READOUT_EVERY = 8           # passes between read-outs: completed accumulations wait in the handle's ring meanwhile
STEP_TARGET_MS = 60.0       # passes per step are chosen so that a step lasts about this long
NOMINAL_FP32_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12   # SMs x lanes x 2 flops x max SM clock


def chain_flops_per_sample(nchan, ntaps, pfb):
    """nominal flops per dual-pol time sample: FFT 5 log2 N per pol, FIR 4T per pol,
    Stokes + accumulate 16."""
    return 10.0 * math.log2(nchan) + (8.0 * ntaps if pfb else 0.0) + 16.0


def kernel_flops_per_sample(cls, nchan, n1, ntaps, pfb):
    n2 = nchan // n1
    if cls == "single":
        return chain_flops_per_sample(nchan, ntaps, pfb)
    if cls == "passA":
        return 10.0 * math.log2(n1) + (8.0 * ntaps if pfb else 0.0)
    if cls == "passB":
        return 10.0 * math.log2(n2) + 16.0
    return 0.0


def world():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def max_over_ranks(x, dist, device):
    """max of a python float over all ranks (identity when not distributed)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return x
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ts, line in self.rows:
            if ts < t0 or ts > t1 + 0.2:
                continue
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0]))
                smax = float(f[1])
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:  # region shorter than the sampling period: take the nearest sample
            for ts, line in self.rows[-3:]:
                try:
                    f = [x.strip() for x in line.split(",")]
                    sm.append(float(f[0]))
                    smax = float(f[1])
                except (ValueError, IndexError):
                    pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm)}


def workload_from_args(a):
    pfb = a.mode == "pfb"
    nchan = a.nchan
    ntaps = 8 if pfb else 1
    chunk_samples = CHUNK_BYTES // 4
    nacc = a.nacc if a.nacc else (256 if nchan == 32768 and pfb else max(1, chunk_samples // a.nsub // nchan // 2))
    name = ("configs[1]: dual-pol PFB N=32768 T=8 M=256, 64 MiB calls" if (pfb and nchan == 32768 and nacc == 256 and a.nsub == 1)
            else f"dual-pol {'PFB T=8' if pfb else 'direct FFT'} N={nchan} M={nacc}, 64 MiB calls"
                 + (f", {a.nsub} interleaved sub-bands (value = dual-pol samples/s summed over the sub-bands)" if a.nsub > 1 else ""))
    return dict(pfb=pfb, nchan=nchan, ntaps=ntaps, nacc=nacc, chunk_samples=chunk_samples, name=name)


def _oracle_stretch(args):
    """Times the oracle as it stands on one stretch of the workload stream (runs in a worker process)."""
    N, T, pfb, nacc, start, budget_s = args
    import oracle
    from paper_1411_0436_b200 import synth
    o = oracle.Oracle(N, T, 2, oracle.MODE_PFB if pfb else oracle.MODE_FFT, nacc,
                      oracle.WINDOW_HANN if pfb else oracle.WINDOW_RECT)
    blocks_per_call = max(1, (1 << 19) // N)
    pos, t_used = start, 0.0
    while t_used < budget_s:
        raw = synth.dual_pol_stream(synth.SEED_BASE + 1, blocks_per_call * N, [synth.F_CFG1], start=pos)
        t0 = time.perf_counter()
        o.process(raw)
        t_used += time.perf_counter() - t0
        pos += blocks_per_call * N
        while o.pending():
            o.read_accum()
    spectra = o.spectra_done()
    o.close()
    return spectra, pos - start, t_used


def cpu_baseline(w, budget_s=10.0, all_cores=True):
    """The oracle as it stands on a bounded prefix of the same stream: one core, and (all_cores) one independent
    stretch of the stream per hardware thread in separate processes (the oracle keeps one static table per process)."""
    N, T = w["nchan"], w["ntaps"]
    spectra, nsamp, t_used = _oracle_stretch((N, T, w["pfb"], w["nacc"], 0, budget_s))
    ghz = spectra * N / t_used / 1e9
    out = {"value": ghz, "unit": "GHz", "cores": 1, "kind": "oracle",
           "sample": f"first {nsamp} time samples ({spectra} spectra) of the workload stream, {t_used:.1f} s of CPU time"}
    if all_cores:
        import concurrent.futures as cf
        import multiprocessing as mp
        ncpu = os.cpu_count() or 1
        try:
            ncpu = len(os.sched_getaffinity(0))
        except (AttributeError, OSError):
            pass
        stride = 1 << 26    # each worker takes its own stretch of the stream
        jobs = [(N, T, w["pfb"], w["nacc"], i * stride, budget_s * 0.6) for i in range(ncpu)]
        t0 = time.perf_counter()
        with cf.ProcessPoolExecutor(max_workers=ncpu, mp_context=mp.get_context("spawn")) as ex:
            res = list(ex.map(_oracle_stretch, jobs))
        wall = time.perf_counter() - t0
        tot_spectra = sum(r[0] for r in res)
        tmax = max(r[2] for r in res)
        out["all_cores"] = {"value": tot_spectra * N / tmax / 1e9, "unit": "GHz", "cores": ncpu, "kind": "oracle",
                            "sample": f"{ncpu} processes, each {budget_s * 0.6:.0f} s on its own 2^26-sample stretch "
                                      f"({tot_spectra} spectra in all; slowest worker {tmax:.1f} s, wall {wall:.1f} s)"}
    return out


def run_reference(a):
    rank, _, ws = world()
    if rank != 0:
        return
    w = workload_from_args(a)
    vals = []
    for _ in range(a.warmup):
        cpu_baseline(w, budget_s=1.0, all_cores=False)
    for _ in range(a.steps):
        vals.append(cpu_baseline(w, budget_s=max(2.0, 40.0 / max(1, a.steps)), all_cores=False))
    v = float(np.mean([x["value"] for x in vals]))
    N = w["nchan"]
    out = {
        "impl": "reference", "metric": "sustained dual-pol bandwidth", "value": v, "unit": "GHz", "n_gpus": a.gpus,
        "steps": a.steps, "warmup": a.warmup, "ms_per_step": None, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w["name"], "nchan": N, "ntaps": w["ntaps"], "npol": 2, "nacc": w["nacc"]},
        "cpu_baseline": {"value": v, "unit": "GHz", "cores": 1, "kind": "oracle", "sample": vals[-1]["sample"]},
        "e2e": {"value": v, "unit": "GHz", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out))


def _setup_device():
    import torch
    rank, local_rank, ws = world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    dist = None
    if ws > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
    return torch, rank, local_rank, ws, device, dist


def _peaks():
    ppath = os.path.join(ROOT, "MEASURED_PEAKS.json")
    return json.load(open(ppath)) if os.path.exists(ppath) else {}


def run_ours(a):
    from paper_1411_0436_b200 import spec as sp
    from paper_1411_0436_b200 import synth

    torch, rank, local_rank, ws, device, dist = _setup_device()

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    w = workload_from_args(a)
    N, T, M, pfb = w["nchan"], w["ntaps"], w["nacc"], w["pfb"]
    cs = w["chunk_samples"]
    pass_samples = cs * CALLS_PER_PASS
    READOUT_EVERY = a.readout_every

    # synthetic stream of configs[1] (config-1 generator), one pass long, per-rank seed
    raw = synth.dual_pol_stream(synth.SEED_BASE + 1 + 1000 * rank, pass_samples, [synth.F_CFG1])
    h_pinned = torch.from_numpy(raw.reshape(-1)).pin_memory()
    d_in = h_pinned.to(device, non_blocking=False)
    stream = torch.cuda.current_stream().cuda_stream

    K = a.nsub                     # eight-sub-band modes: the same bytes are K interleaved sub-bands of cs / K time samples
    cs //= K
    pass_samples //= K
    s = sp.Spec(N, T, 2, sp.MODE_PFB if pfb else sp.MODE_FFT, M, sp.WINDOW_HANN if pfb else sp.WINDOW_RECT, nsub=K)
    if a.tensor_core_stage:
        s.set_option(sp.OPT_TENSOR_CORE_STAGE, 1)
    n1, n2, plan_desc = s.plan_info()
    if a.tensor_core_stage:
        plan_desc += " [first 16-point DFT factor on the tensor cores: tcgen05.mma]"
    # accumulations are read out once per READOUT_EVERY passes (32 calls), so that consecutive spec_process launches
    # stay adjacent in the stream and may overlap; the ring holds what completes meanwhile
    ring = max(8, READOUT_EVERY * CALLS_PER_PASS * (cs // N // M + 1) + 2)
    s.set_ring(ring)
    d_out = torch.empty((ring, K * 4, N), dtype=torch.float32, device=device)
    fp32_peak = sp.measure_fp32_peak(stream)

    npass = [0]
    last_batch = [0]

    def pass_resident():
        nout = 0
        for c in range(CALLS_PER_PASS):
            s.process(d_in.data_ptr() + c * cs * 4 * K, cs, stream)
        npass[0] += 1
        if npass[0] % READOUT_EVERY == 0:
            while s.pending():
                last_batch[0] = s.read_accum_batch_device(d_out.data_ptr(), ring, stream)
                nout += last_batch[0]
        return nout

    def selfcheck(nout_timed, passes, steps):
        """After the timed region, outside it, without the oracle (tests/ holds the parity tests of this very call
        pattern): (1) the number of accumulations read out is the one the samples fed amount to; (2) every pass feeds
        the same bytes and the filter history carries over, so the integrated spectra repeat with the period at which
        pass and accumulation boundaries realign: the last read-out batch must agree with itself shifted by that
        period, to fp32 summation order (the partial sums meet in HBM by atomics, in no fixed order)."""
        spectra_per_pass = pass_samples // N
        expected = steps * passes * spectra_per_pass / M
        res = {"records": int(nout_timed), "records_expected": expected, "ok": abs(nout_timed - expected) <= 1.0}
        n = last_batch[0]
        period = spectra_per_pass // math.gcd(spectra_per_pass, M) if pass_samples % N == 0 else 0
        if period and n > period:
            x, y = d_out[:n - period], d_out[period:n]
            scale = x.abs().amax().item()
            err = ((x - y).abs().amax().item() / scale) if scale > 0 else float("inf")
            finite = bool(torch.isfinite(d_out[:n]).all().item())
            res.update({"period_records": period, "records_compared": n - period, "repeat_rel_err": err,
                        "finite": finite, "ok": res["ok"] and finite and err < 1e-4})
        return res

    # e2e read-back: completed accumulations are popped into one of two device buffers and copied to pinned host
    # memory on a third stream, so that the device-to-host copy of pass i overlaps the host-to-device copies and the
    # kernels of pass i+1 (the host link is full duplex)
    d2h = torch.cuda.Stream(device=device)
    ring_e = max(8, CALLS_PER_PASS * (cs // N // M + 1) + 2)
    d_oute = [torch.empty((ring_e, K * 4, N), dtype=torch.float32, device=device) for _ in range(2)]
    h_oute = [torch.empty((ring_e, K * 4, N), dtype=torch.float32).pin_memory() for _ in range(2)]
    ev_popped = [torch.cuda.Event() for _ in range(2)]
    ev_copied = [torch.cuda.Event() for _ in range(2)]
    epass = [0]

    def pass_e2e():
        k = epass[0] & 1
        epass[0] += 1
        main = torch.cuda.current_stream()
        s.stream_host(h_pinned.data_ptr(), pass_samples, cs, stream)
        main.wait_event(ev_copied[k])            # buffer k's previous contents have reached the host
        nout = 0
        while s.pending() and nout < ring_e:
            nout += s.read_accum_batch_device(d_oute[k].data_ptr() + nout * 16 * N * K, ring_e - nout, stream)
        ev_popped[k].record(main)
        d2h.wait_event(ev_popped[k])
        with torch.cuda.stream(d2h):
            h_oute[k][:nout].copy_(d_oute[k][:nout], non_blocking=True)
            ev_copied[k].record(d2h)
        return nout

    def drain():
        while s.pending():
            s.read_accum_batch_device(d_out.data_ptr(), ring, stream)
        npass[0] = 0

    def one_pass_ms(fn, reps=3):
        for _ in range(reps):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    def timed(fn, passes, steps, warmup, profile):
        drain()
        for _ in range(warmup):
            for _ in range(passes):
                fn()
        barrier()
        s.profile(profile)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.time()
        e0.record()
        nout = 0
        for _ in range(steps):
            for _ in range(passes):
                nout += fn()
        torch.cuda.current_stream().wait_stream(d2h)   # (e2e: the last read-back is inside the timed region)
        e1.record()
        barrier()
        t1 = time.time()
        ms = max_over_ranks(e0.elapsed_time(e1), dist, device)
        return ms, nout, s.profile_read(), (t0, t1)

    # passes per step: fixed before the timed region from a short calibration (the same on every rank); a whole
    # number of read-out intervals, so that every step carries its own read-outs
    p_res = max(1, int(math.ceil(STEP_TARGET_MS / max_over_ranks(one_pass_ms(pass_resident, READOUT_EVERY), dist, device))))
    p_res = ((p_res + READOUT_EVERY - 1) // READOUT_EVERY) * READOUT_EVERY
    p_e2e = max(1, int(math.ceil(STEP_TARGET_MS / max_over_ranks(one_pass_ms(pass_e2e, 1), dist, device))))

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    ms, nout, prof0, (t0, t1) = timed(pass_resident, p_res, a.steps, a.warmup, False)
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    try:
        check = selfcheck(nout, p_res, a.steps)
    except Exception as e:                       # the check must never cost the measurement
        check = {"ok": None, "error": repr(e)}
    # per-kernel split: the same passes again with every launch bracketed by CUDA events (kept out of the pass
    # above: the event records cost device time and keep consecutive launches from overlapping)
    prof_steps = max(1, min(a.steps, 4))
    ms_prof, _, prof, _ = timed(pass_resident, p_res, prof_steps, 1, True)
    ms_e2e, nout_e2e, prof_e2e, _ = timed(pass_e2e, p_e2e, a.steps, max(1, a.warmup // 2), False)
    s.close()

    step_samples = pass_samples * p_res * K        # dual-pol samples over all sub-bands
    total_samples = step_samples * a.steps * ws
    value = total_samples / (ms * 1e-3) / 1e9
    e2e_step_samples = pass_samples * p_e2e * K
    e2e = e2e_step_samples * a.steps * ws / (ms_e2e * 1e-3) / 1e9

    # dominant kernel and its roofline (per-launch averages)
    kern = max(("single", "passA", "passB"), key=lambda k: prof[k][0])
    k_ms, k_n = prof[kern]                       # event-bracketed pass (prof_steps steps)
    launches0 = {k: v[1] for k, v in prof0.items()}   # launch counts of the timed pass
    kern_name = plan_desc if kern == "single" else f"{kern} of: {plan_desc}"
    fps = kernel_flops_per_sample(kern, N, n1, T, pfb)
    frac_bracketed = (fps * step_samples * prof_steps / (k_ms * 1e-3) / 1e12 / fp32_peak) if k_ms > 0 else None
    readout_ms = prof["readout"][0] / prof_steps * a.steps        # read-out kernels' share of the timed pass
    one_kernel = (kern == "single")
    if one_kernel and ms > readout_ms and launches0[kern]:
        ms_per_launch = (ms - readout_ms) / launches0[kern]
        achieved = fps * step_samples * a.steps / ((ms - readout_ms) * 1e-3) / 1e12
        timing = ("timed pass itself: (step time - read-out kernels) / launches; consecutive launches overlap "
                  "there (programmatic dependent launch), no event sits between them")
    else:
        ms_per_launch = k_ms / k_n if k_n else None
        achieved = frac_bracketed * fp32_peak if frac_bracketed else None
        timing = "CUDA events around every launch of a second pass over the same steps (several kernels share the step)"
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        traffic = json.load(open(tpath)).get(f"{kern}:{'pfb' if pfb else 'fft'}:{N}")
    hbm = _peaks().get("hbm_gbs", 6650.0)
    F = chain_flops_per_sample(N, T, pfb)
    roof_ghz = min(hbm / 4.0, fp32_peak * 1e3 / F)
    launches = sum(launches0.values())

    if rank != 0:
        return
    out = {
        "metric": "sustained dual-pol bandwidth", "value": value, "unit": "GHz", "n_gpus": ws, "steps": a.steps,
        "warmup": a.warmup, "ms_per_step": ms / a.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w["name"], "nchan": N, "ntaps": T, "npol": 2, "nacc": M, "mode": a.mode,
                   "samples_per_step": step_samples, "calls_per_step": CALLS_PER_PASS * p_res,
                   "passes_per_step": p_res, "timed_region_s": ms * 1e-3,
                   "cache": "every pass streams 256 MiB of input > 126 MB L2 (no flush needed)",
                   "readout": f"spec_read_accum_batch every {READOUT_EVERY} passes ({READOUT_EVERY * CALLS_PER_PASS} calls), inside the timed region",
                   "plan": plan_desc,
                   "parallelism": f"replicas x{ws}" if ws > 1 else "single GPU",
                   "paper_context": "GTX TITAN: 1.1 GHz (PFB) / 1.4 GHz (FFT) dual-pol, PAPER.md:7"},
        "e2e": {"value": e2e, "unit": "GHz", "h2d_bytes_per_step": e2e_step_samples * 4,
                "d2h_bytes_per_step": int(nout_e2e / a.steps * 16 * N * K), "ms_per_step": ms_e2e / a.steps,
                "passes_per_step": p_e2e, "h2d_gbs": e2e_step_samples * 4 * a.steps / (ms_e2e * 1e-3) / 1e9},
        "gpu_launches": int(launches),
        "selfcheck": check,
        "clocks": clocks,
        "roofline": {"bound": "alu", "kernel": kern, "kernel_name": kern_name, "achieved": achieved, "peak": fp32_peak,
                     "unit": "TFLOP/s", "frac": (achieved / fp32_peak) if achieved else None, "traffic": traffic,
                     "traffic_note": "dram bytes read+write per launch from the ncu --set full capture listed in "
                                     "profiles/traffic.json (algorithmic: 4 B per dual-pol sample)",
                     "algorithmic_bytes_per_launch": 4 * cs,
                     "launches_note": (f"{K} sub-bands: one launch per sub-band and call, {cs} samples each" if K > 1 else None),
                     "peak_source": "spec_measure_fp32_peak in this run (FFMA chains, all SMs); "
                                    "MEASURED_PEAKS.json has no fp32 figure",
                     "peak_nominal": NOMINAL_FP32_TFLOPS, "launches": int(launches0[kern]),
                     "ms_per_launch": ms_per_launch, "timing": timing,
                     "frac_event_bracketed": frac_bracketed,
                     "kernel_ms_event_bracketed": {k: v[0] / prof_steps for k, v in prof.items()},
                     "ms_per_step_event_bracketed": ms_prof / prof_steps},
        "roofline_chain": {"flops_per_sample": F, "hbm_bound_ghz": hbm / 4.0, "fp32_bound_ghz": fp32_peak * 1e3 / F,
                           "roof_ghz": roof_ghz, "frac": value / ws / roof_ghz},
    }
    if ws == 1 and not a.no_cpu:
        out["cpu_baseline"] = cpu_baseline(w)
    print(json.dumps(out))
    if check["ok"] is not True:
        print(f"bench.py: self-check FAILED, the number above is not valid: {check}", file=sys.stderr)
    if dist is not None:
        dist.destroy_process_group()


def run_sweep(a):
    """configs[4]: N = 2^10 .. 2^19 x {PFB T=8, direct FFT}, dual-pol full Stokes, nacc chosen so that each run
    processes 2^L time samples of the config-1 generator (L = 31 by default: nacc = 2^31/N, minus 7 for the PFB),
    once device-resident and once streamed from pinned host memory with double buffering.  The 2^L samples are
    the 2^26-sample device / pinned buffer fed repeatedly (the 8 GiB stream itself would take minutes to draw)."""
    from paper_1411_0436_b200 import spec as sp
    from paper_1411_0436_b200 import synth

    torch, rank, local_rank, ws, device, dist = _setup_device()
    if rank != 0:
        return
    L = a.sweep_log2
    buf_samples = 1 << min(26, L)
    reps = (1 << L) // buf_samples
    cs = CHUNK_BYTES // 4
    raw = synth.dual_pol_stream(synth.SEED_BASE + 4, buf_samples, [synth.F_CFG1])
    h_pinned = torch.from_numpy(raw.reshape(-1)).pin_memory()
    d_in = h_pinned.to(device)
    stream = torch.cuda.current_stream().cuda_stream
    t_warm = time.time()
    while time.time() - t_warm < 1.5:      # bring the clocks up before the first point (the GPU was idle until now)
        fp32_peak = sp.measure_fp32_peak(stream)
    hbm = _peaks().get("hbm_gbs", 6650.0)
    rows = []
    for mode in ("fft", "pfb"):
        for lg in range(10, 20):
            N = 1 << lg
            pfb = mode == "pfb"
            T = 8 if pfb else 1
            M = (1 << L) // N - (T - 1)
            s = sp.Spec(N, T, 2, sp.MODE_PFB if pfb else sp.MODE_FFT, M, sp.WINDOW_HANN if pfb else sp.WINDOW_RECT)
            d_out = torch.empty((4, N), dtype=torch.float32, device=device)

            def run_resident():
                done = 0
                for r in range(reps):
                    for c in range(buf_samples // cs):
                        done += s.process(d_in.data_ptr() + c * cs * 4, cs, stream)
                assert done == 1, done
                assert s.read_accum_device(d_out.data_ptr(), stream) == 1

            def run_streamed():
                done = 0
                for r in range(reps):
                    done += s.stream_host(h_pinned.data_ptr(), buf_samples, cs, stream)
                assert done == 1, done
                assert s.read_accum_host(stream) is not None

            res = {}
            for name, fn, nrep in (("resident", run_resident, a.sweep_reps), ("streamed", run_streamed, 1)):
                for _ in range(2 if name == "resident" else 1):   # warm-up runs
                    s.reset(); fn()
                s.reset()
                times = []
                for _ in range(nrep):
                    torch.cuda.synchronize()
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(); fn(); e1.record()
                    torch.cuda.synchronize()
                    times.append(e0.elapsed_time(e1))
                    s.reset()
                res[name] = (1 << L) / (float(np.median(times)) * 1e-3) / 1e9
                res[name + "_ms"] = [round(t, 3) for t in times]
            _, _, desc = s.plan_info()
            s.close()
            F = chain_flops_per_sample(N, T, pfb)
            roof = min(hbm / 4.0, fp32_peak * 1e3 / F)
            row = {"sweep_point": True, "mode": mode, "nchan": N, "ntaps": T, "nacc": M, "samples": 1 << L,
                   "resident_ghz": res["resident"], "streamed_ghz": res["streamed"], "resident_runs_ms": res["resident_ms"],
                   "streamed_h2d_gbs": res["streamed"] * 4, "roof_ghz": roof, "frac": res["resident"] / roof,
                   "fp32_peak_tflops": fp32_peak, "plan": desc}
            rows.append(row)
            print(json.dumps(row), flush=True)
    print(f"\n| mode | N | nacc | resident GHz | % of roofline | streamed GHz (host link GB/s) | roofline GHz |")
    print("|---|---|---|---|---|---|---|")
    for r in rows:
        print(f"| {r['mode']} | {r['nchan']} | {r['nacc']} | {r['resident_ghz']:.1f} | {100 * r['frac']:.1f} | "
              f"{r['streamed_ghz']:.2f} ({r['streamed_h2d_gbs']:.1f}) | {r['roof_ghz']:.0f} |")
    print(f"\n2^{L} time samples per point (the 2^{min(26, L)}-sample config-1 buffer fed {reps} times), 64 MiB calls; "
          f"roofline = min(HBM {hbm:.0f} GB/s / 4 B, fp32 {fp32_peak:.1f} TFLOP/s measured in this run / F(N)); "
          f"resident: median of {a.sweep_reps} runs.")


def run_packets(a):
    """the real-time ingest shape, many small calls.  A periodic segment of 18
    spec_process calls of 8 blocks each plus its three batched read-outs, issued call by call and as ONE CUDA graph."""
    from paper_1411_0436_b200 import spec as sp
    from paper_1411_0436_b200 import synth
    torch, rank, local_rank, ws, device, dist = _setup_device()
    if rank != 0:
        return
    pfb = a.mode == "pfb"
    N, T, M, bpc, ncalls = a.nchan, (8 if pfb else 1), 16, 8, 18
    seg = bpc * ncalls * N
    raw = synth.dual_pol_stream(synth.SEED_BASE + 5, (T - 1) * N + seg, [synth.F_CFG1])
    d_all = torch.from_numpy(raw.reshape(-1)).to(device)
    d_seg = d_all[(T - 1) * N * 4:]
    d_out = torch.zeros((9, 4, N), dtype=torch.float32, device=device)
    res = {}
    for use_graph in (False, True):
        s = sp.Spec(N, T, 2, sp.MODE_PFB if pfb else sp.MODE_FFT, M, sp.WINDOW_HANN if pfb else sp.WINDOW_RECT)
        if T > 1:
            s.process(d_all.data_ptr(), (T - 1) * N, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()

        def segment(st):
            got = 0
            for c in range(ncalls):
                s.process(d_seg.data_ptr() + c * bpc * N * 4, bpc * N, st)
                if c % 6 == 5:
                    got += s.read_accum_batch_device(d_out.data_ptr() + got * 16 * N, 8, st)
            return got

        if use_graph:
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                s.capture_begin()
                segment(torch.cuda.current_stream().cuda_stream)
                s.capture_end()
            run = g.replay
        else:
            run = lambda: segment(torch.cuda.current_stream().cuda_stream)
        for _ in range(20):
            run()
        torch.cuda.synchronize()
        reps = 200
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record()
        for _ in range(reps):
            run()
        e1.record()
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        ms = e0.elapsed_time(e1)
        res["graph" if use_graph else "calls"] = {"us_per_call_device": ms * 1e3 / (reps * ncalls), "us_per_call_host": wall * 1e6 / (reps * ncalls),
                                                   "ghz": reps * bpc * ncalls * N / (ms * 1e-3) / 1e9}
        s.close()
    print(json.dumps({"packets": True, "mode": a.mode, "nchan": N, "blocks_per_call": bpc, "calls_per_segment": ncalls,
                      "samples_per_call": bpc * N, **res}))


def main():
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=20)
    p.add_argument("--warmup", type=int, default=3)
    p.add_argument("--impl", default="ours", choices=["ours", "reference"])
    p.add_argument("--nchan", type=int, default=32768)
    p.add_argument("--mode", default="pfb", choices=["pfb", "fft"])
    p.add_argument("--nacc", type=int, default=0)
    p.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    p.add_argument("--readout-every", type=int, default=READOUT_EVERY, help="passes between read-outs of the resident arm")
    p.add_argument("--nsub", type=int, default=1, help="eight-sub-band modes (PAPER.md:73): interleaved sub-bands per time sample")
    p.add_argument("--packets", action="store_true",
                   help="NEXT-4: packet-sized calls (8 blocks each), issued one by one and replayed as one CUDA graph")
    p.add_argument("--tensor-core-stage", action="store_true",
                   help="direct-FFT mode, N = 16384 or 32768: first DFT factor via tcgen05.mma (spec_set_option)")
    p.add_argument("--probes", action="store_true", help="instruction-throughput probes quoted in DESIGN.md section 6")
    p.add_argument("--sweep", action="store_true", help="configs[4]: all 20 points, resident and streamed")
    p.add_argument("--sweep-log2", type=int, default=31, help="log2 of the time samples per sweep point")
    p.add_argument("--sweep-reps", type=int, default=3)
    a = p.parse_args()
    if a.tensor_core_stage and (a.mode != "fft" or a.nchan not in (16384, 32768)):
        p.error("--tensor-core-stage needs --mode fft and --nchan 16384 or 32768 (include/spec.h, spec_set_option)")
    if a.warmup < 3 and a.impl == "ours":
        a.warmup = 3
    if a.impl == "reference":
        run_reference(a)
    elif a.probes:
        from paper_1411_0436_b200 import spec as sp
        for _ in range(3):
            sp.measure_fp32_peak(0)      # clocks up
        print(json.dumps({"probes_thread_instructions_per_clk_sm": {n: round(sp.debug_probe(i), 1) for i, n in enumerate(sp.PROBES)}}))
    elif a.packets:
        run_packets(a)
    elif a.sweep:
        run_sweep(a)
    else:
        run_ours(a)


if __name__ == "__main__":
    main()

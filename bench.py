#!/usr/bin/env python
"""bench.py — sustained dual-pol bandwidth of the spectrometer hot path on B200.

Metric (BASELINE.json): complex samples/s per polarisation (= per-polarisation bandwidth) in GHz,
PFB mode by default on configs[1]: dual-pol PFB, N=32768, T=8, M=256, fed in 64 MiB calls that carry
the 7*N filter history.  One "step" = 4 such calls (2^26 time samples, 256 MiB of int8 input, larger
than the 126 MB L2) through the whole chain unpack -> FIR -> FFT -> Stokes -> accumulate -> read-out.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                  [--nchan N --mode pfb|fft --nacc M]   (other sweep points, same JSON line)

`value`  : inputs resident in HBM before the timed region.
`e2e`    : the same work through spec_stream_host from PINNED HOST memory (H2D inside the timed
           region, double-buffered on a side stream) plus a device-to-host read of every completed
           accumulation.
`roofline`: dominant kernel's nominal fp32 flops / its CUDA-event time vs the fp32 peak measured in
           this run (spec_measure_fp32_peak); `roofline_chain` is north_star's whole-chain roofline.
`cpu_baseline`: the CPU oracle (oracle/, fp64, single thread) timed on a bounded sample.
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
CALLS_PER_STEP = 4
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


def four_step_split(nchan):
    if nchan <= 4096:
        return 1
    return 16 if nchan <= 65536 else nchan // 4096


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
    nacc = a.nacc if a.nacc else (256 if nchan == 32768 and pfb else max(1, chunk_samples // nchan // 2))
    name = ("configs[1]: dual-pol PFB N=32768 T=8 M=256, 64 MiB calls" if (pfb and nchan == 32768 and nacc == 256)
            else f"dual-pol {'PFB T=8' if pfb else 'direct FFT'} N={nchan} M={nacc}, 64 MiB calls")
    return dict(pfb=pfb, nchan=nchan, ntaps=ntaps, nacc=nacc, chunk_samples=chunk_samples, name=name)


def cpu_baseline(w, budget_s=10.0):
    """The oracle as it stands, single thread, on a bounded prefix of the same stream."""
    import oracle
    from paper_1411_0436_b200 import synth
    N, T = w["nchan"], w["ntaps"]
    o = oracle.Oracle(N, T, 2, oracle.MODE_PFB if w["pfb"] else oracle.MODE_FFT, w["nacc"],
                      oracle.WINDOW_HANN if w["pfb"] else oracle.WINDOW_RECT)
    blocks_per_call = max(1, (1 << 19) // N)
    pos, spectra, t_used = 0, 0, 0.0
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
    ghz = spectra * N / t_used / 1e9
    return {"value": ghz, "unit": "GHz", "cores": 1, "kind": "oracle",
            "sample": f"first {pos} time samples ({spectra} spectra) of the workload stream, {t_used:.1f} s of CPU time"}


def run_reference(a):
    rank, _, ws = world()
    if rank != 0:
        return
    w = workload_from_args(a)
    vals = []
    for _ in range(a.warmup):
        cpu_baseline(w, budget_s=1.0)
    for _ in range(a.steps):
        vals.append(cpu_baseline(w, budget_s=max(2.0, 40.0 / max(1, a.steps))))
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


def run_ours(a):
    import torch

    from paper_1411_0436_b200 import spec as sp
    from paper_1411_0436_b200 import synth

    rank, local_rank, ws = world()
    dist = None
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    if ws > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    w = workload_from_args(a)
    N, T, M, pfb = w["nchan"], w["ntaps"], w["nacc"], w["pfb"]
    cs = w["chunk_samples"]
    step_samples = cs * CALLS_PER_STEP
    n1 = four_step_split(N)

    # synthetic stream of configs[1] (config-1 generator), one step long, per-rank seed
    raw = synth.dual_pol_stream(synth.SEED_BASE + 1 + 1000 * rank, step_samples, [synth.F_CFG1])
    h_pinned = torch.from_numpy(raw.reshape(-1)).pin_memory()
    d_in = h_pinned.to(device, non_blocking=False)
    stream = torch.cuda.current_stream().cuda_stream

    s = sp.Spec(N, T, 2, sp.MODE_PFB if pfb else sp.MODE_FFT, M, sp.WINDOW_HANN if pfb else sp.WINDOW_RECT)
    # accumulations are read out once per step (after its CALLS_PER_STEP calls), so that consecutive
    # spec_process launches stay adjacent in the stream and may overlap
    ring = max(8, CALLS_PER_STEP * (cs // N // M + 1) + 2)
    s.set_ring(ring)
    d_out = torch.empty((ring, 4, N), dtype=torch.float32, device=device)
    fp32_peak = sp.measure_fp32_peak(stream)

    def step_resident():
        nout = 0
        for c in range(CALLS_PER_STEP):
            s.process(d_in.data_ptr() + c * cs * 4, cs, stream)
        while s.pending():
            nout += s.read_accum_batch_device(d_out.data_ptr(), ring, stream)
        return nout

    def step_e2e():
        nout = 0
        s.stream_host(h_pinned.data_ptr(), step_samples, cs, stream)
        while s.pending():
            s.read_accum_host(stream)
            nout += 1
        return nout

    def timed(fn, steps, warmup, profile):
        for _ in range(warmup):
            fn()
        barrier()
        s.profile(profile)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.time()
        e0.record()
        nout = 0
        for _ in range(steps):
            nout += fn()
        e1.record()
        barrier()
        t1 = time.time()
        ms = max_over_ranks(e0.elapsed_time(e1), dist, device)
        return ms, nout, s.profile_read(), (t0, t1)

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    ms, nout, prof0, (t0, t1) = timed(step_resident, a.steps, a.warmup, False)
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    # per-kernel split for the roofline: the same K steps again with every launch bracketed by CUDA
    # events (kept out of the pass above: the event records themselves cost device time)
    ms_prof, _, prof, _ = timed(step_resident, a.steps, 1, True)
    ms_e2e, nout_e2e, prof_e2e, _ = timed(step_e2e, a.steps, max(1, a.warmup // 2), False)
    s.close()

    total_samples = step_samples * a.steps * ws
    value = total_samples / (ms * 1e-3) / 1e9
    e2e = total_samples / (ms_e2e * 1e-3) / 1e9

    # dominant kernel and its roofline (per-launch averages over the timed region)
    kern = max(("single", "passA", "passB"), key=lambda k: prof[k][0])
    k_ms, k_n = prof[kern]
    fused = (pfb and 1024 <= N <= 65536) or (not pfb and 8192 <= N <= 65536)
    kern_name = {"single": "k_fused (persistent four-step: unpack+FIR+FFT+Stokes+accumulate)" if fused
                 else "k_engine (single-CTA unpack+window+FFT+Stokes+accumulate)",
                 "passA": "four-step pass A", "passB": "four-step pass B"}[kern]
    flops_total = kernel_flops_per_sample(kern, N, n1, T, pfb) * step_samples * a.steps
    achieved = flops_total / (k_ms * 1e-3) / 1e12 if k_ms > 0 else None
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        traffic = json.load(open(tpath)).get(f"{kern}:{'pfb' if pfb else 'fft'}:{N}")
    peaks = {}
    ppath = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(ppath):
        peaks = json.load(open(ppath))
    hbm = peaks.get("hbm_gbs", 6650.0)
    F = chain_flops_per_sample(N, T, pfb)
    roof_ghz = min(hbm / 4.0, fp32_peak * 1e3 / F)
    launches = sum(v[1] for v in prof0.values())

    if rank != 0:
        return
    out = {
        "metric": "sustained dual-pol bandwidth", "value": value, "unit": "GHz", "n_gpus": ws, "steps": a.steps,
        "warmup": a.warmup, "ms_per_step": ms / a.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w["name"], "nchan": N, "ntaps": T, "npol": 2, "nacc": M, "mode": a.mode,
                   "samples_per_step": step_samples, "calls_per_step": CALLS_PER_STEP,
                   "cache": "input per step 256 MiB > 126 MB L2 (no flush needed)", "readout": "spec_read_accum_batch after every step (its 4 calls), inside the timed region",
                   "parallelism": f"replicas x{ws}" if ws > 1 else "single GPU",
                   "paper_context": "GTX TITAN: 1.1 GHz (PFB) / 1.4 GHz (FFT) dual-pol, PAPER.md:7"},
        "e2e": {"value": e2e, "unit": "GHz", "h2d_bytes_per_step": step_samples * 4,
                "d2h_bytes_per_step": int(nout_e2e / a.steps * 16 * N), "ms_per_step": ms_e2e / a.steps,
                "h2d_gbs": step_samples * 4 * a.steps / (ms_e2e * 1e-3) / 1e9},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": {"bound": "alu", "kernel": kern, "kernel_name": kern_name, "achieved": achieved, "peak": fp32_peak, "unit": "TFLOP/s",
                     "frac": (achieved / fp32_peak) if achieved else None, "traffic": traffic,
                     "traffic_note": "dram bytes read+write per launch from the ncu --set full capture listed in "
                                     "profiles/traffic.json (algorithmic: 4 B per dual-pol sample)",
                     "algorithmic_bytes_per_launch": 4 * step_samples // CALLS_PER_STEP,
                     "peak_source": "spec_measure_fp32_peak in this run (FFMA chains, all SMs); "
                                    "MEASURED_PEAKS.json has no fp32 figure",
                     "peak_nominal": NOMINAL_FP32_TFLOPS, "launches": int(k_n),
                     "ms_per_launch": k_ms / k_n if k_n else None,
                     "kernel_ms": {k: v[0] for k, v in prof.items()},
                     "timing": "CUDA events around every launch of a second pass over the same K steps "
                               f"({ms_prof / a.steps:.3f} ms/step with the events in the stream)",
                     # consecutive k_fused launches overlap in the un-bracketed stream (programmatic dependent
                     # launch); the events of the second pass serialise them, so `frac` is the conservative figure.
                     # Where one kernel is the whole chain, this is the same ratio from the first (timed) pass:
                     # its total time minus the read-out kernels' time of the second pass
                     "frac_in_stream": (flops_total / ((ms - prof["readout"][0]) * 1e-3) / 1e12 / fp32_peak)
                     if (kern == "single" and ms > prof["readout"][0]) else None},
        "roofline_chain": {"flops_per_sample": F, "hbm_bound_ghz": hbm / 4.0, "fp32_bound_ghz": fp32_peak * 1e3 / F,
                           "roof_ghz": roof_ghz, "frac": value / ws / roof_ghz},
    }
    if ws == 1 and not a.no_cpu:
        out["cpu_baseline"] = cpu_baseline(w)
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def main():
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=10)
    p.add_argument("--warmup", type=int, default=3)
    p.add_argument("--impl", default="ours", choices=["ours", "reference"])
    p.add_argument("--nchan", type=int, default=32768)
    p.add_argument("--mode", default="pfb", choices=["pfb", "fft"])
    p.add_argument("--nacc", type=int, default=0)
    p.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    a = p.parse_args()
    if a.warmup < 3 and a.impl == "ours":
        a.warmup = 3
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)


if __name__ == "__main__":
    main()

"""The N>1 path of bench.py on CPU: two gloo ranks (world_size 2, rendezvous on 127.0.0.1).
The spectrometer shards over independent streams (one beam per GPU):
no data-path collective, only the max-over-ranks of the elapsed time and per-rank input seeds."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys, json
    sys.path.insert(0, %r)
    import numpy as np
    import torch
    import torch.distributed as dist
    import bench
    from paper_1411_0436_b200 import synth
    dist.init_process_group("gloo")
    rank, ws = dist.get_rank(), dist.get_world_size()
    assert bench.world()[0] == rank and bench.world()[2] == ws
    # max over ranks of a per-rank time: rank r reports 10 + r
    t = bench.max_over_ranks(10.0 + rank, dist, torch.device("cpu"))
    # per-rank streams differ (independent beams) and are reproducible
    raw = synth.dual_pol_stream(synth.SEED_BASE + 1 + 1000 * rank, 4096, [synth.F_CFG1])
    digest = int(np.abs(raw.astype(np.int64)).sum())
    out = [None] * ws
    dist.all_gather_object(out, (t, digest))
    if rank == 0:
        print(json.dumps(out))
    dist.destroy_process_group()
""")


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def test_two_gloo_ranks_max_time_and_independent_streams(tmp_path):
    import json
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=120) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e
    res = json.loads(outs[0][0].strip().splitlines()[-1])
    assert [r[0] for r in res] == [11.0, 11.0]          # both ranks see the slower rank's time
    assert res[0][1] != res[1][1]                        # different beams, different bytes
    assert outs[1][0].strip() == ""                      # only rank 0 prints


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""

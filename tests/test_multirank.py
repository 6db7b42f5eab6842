"""N > 1 path of bench.py on CPU (gloo, world_size 2): replicas only -- every rank runs the whole hot path on
its own batch, the only cross-rank step is the MAX over ranks of the device-timed durations (DESIGN.md
section 1, row e).  Also: `bench.py --impl reference` under a 2-rank launch prints exactly one line."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    from pvf_inputs import make_events
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ev = make_events("run3", 6, bench.rank_seed("run3", rank))
    ms, ms_e2e = bench.max_over_ranks([10.0 + 5.0 * rank, 30.0 - rank], dist, "cpu")
    out[rank] = (int(ev.n_tracks), float(ev.feat[0, 0]), ms, ms_e2e)
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_and_max_over_ranks():
    import torch.multiprocessing as mp
    port = _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        r0, r1 = out[0], out[1]
    assert (r0[0], r0[1]) != (r1[0], r1[1])            # each replica has its own batch
    assert r0[2] == r1[2] == 15.0 and r0[3] == r1[3] == 30.0   # MAX over ranks, identical on all ranks
    sys.path.insert(0, ROOT)
    import bench
    assert bench.whole_job_rate(2, 16000, 5, 100.0) == pytest.approx(2 * 16000 * 5 / 0.1)


def test_reference_arm_prints_one_line_under_two_ranks():
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--steps", "1", "--warmup", "0", "--ref-sample", "2", "--events", "4"]
    env = dict(os.environ, OMP_NUM_THREADS="2")
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT, env=env)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0

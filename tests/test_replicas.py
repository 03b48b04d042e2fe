"""Multi-rank host logic of bench.py (replicas: one independent configuration per GPU) at world size 2
over gloo on the CPU, and the reference arm under torchrun (rank 0 alone works and prints)."""
import json
import os
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    import ensembles as E
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = dict(E.CONFIGS["C0"])
    U, _ = bench.make_links("C0", rank)                       # rank r: its own configuration of the same ensemble
    ms_local = 10.0 * (rank + 1)                              # rank 1 is the slow one
    ms = bench.max_over_ranks(ms_local, dist, "cpu")
    dist.barrier()
    out[rank] = (bench.rank_stream(cfg, rank), float(np.abs(U).sum()), ms, bench.whole_job_value(world, 5, 100, ms))
    dist.destroy_process_group()


def test_replicas_world_size_2_gloo():
    import torch.multiprocessing as mp
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        r0, r1 = out[0], out[1]
    assert r0[0] != r1[0] and r0[1] != r1[1]                  # different Philox streams, different links
    assert r0[2] == r1[2] == 20.0                             # both ranks see the slowest rank's time
    assert r0[3] == r1[3] == 2 * 5 * 100 / 0.020              # whole-job iterations/s


def test_reference_arm_under_torchrun_prints_once():
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--workload", "C0"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                    # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["n_gpus"] == 2

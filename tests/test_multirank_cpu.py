"""N>1 host logic on CPU (gloo, world_size 2): the path shards by independent batches (weak scaling, no data-path
collective), so what there is to test is the per-rank batch selection, the max-over-ranks timing reduction, the
whole-job throughput arithmetic and that only rank 0 of the reference arm prints."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import bench
    import tqp_inputs as ti
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 * (rank + 1), dist, torch.device("cpu"))
    cfg = bench.rank_config(ti.CONFIGS[0], rank)
    x = ti.make_inputs(cfg)["X"]
    gathered = [None] * world
    dist.all_gather_object(gathered, int(np.asarray(x, np.int64).sum()))
    out[rank] = (ms, cfg.seed, gathered)
    dist.destroy_process_group()


def test_gloo_two_ranks_timing_and_batches():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == 20.0 and res[1][0] == 20.0              # max over ranks, same on every rank
    assert res[0][1] != res[1][1]                               # independent batches
    assert res[0][2][0] != res[0][2][1]                         # ... with different contents
    import bench
    assert bench.whole_job_value(2, 8192, 20, 100.0) == 2 * 8192 * 20 / 0.1


def test_reference_arm_prints_once_under_torchrun():
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--config", "0", "--ref-tokens", "16"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["cpu_baseline"]["kind"] == "oracle" and j["value"] > 0
    assert j["e2e"]["h2d_bytes_per_step"] == 0 and j["n_gpus"] == 2

"""N > 1 host logic on CPU (gloo, world_size 2): independent per-rank batches (no data-path
collective), max-over-ranks timing, whole-job throughput."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from harness import workloads as W
    wl = W.make(1, seed=bench.rank_seed(42, rank))
    toks, off = wl.queue.materialize_np()
    ms = bench.max_over_ranks(10.0 * (rank + 1), torch.device("cpu"), world)
    # every rank's batch has the same shape but different content
    digest = torch.tensor([float(int(toks[:1000].astype(np.int64).sum()))], dtype=torch.float64)
    all_d = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(all_d, digest)
    out[rank] = (ms, wl.N, [float(d.item()) for d in all_d], bench.job_throughput(wl.N, world, 4, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_world2_independent_batches_and_max_timing():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    assert set(out.keys()) == {0, 1}
    for r in range(world):
        ms, n, digests, thr = out[r]
        assert ms == 20.0                      # max over ranks, identical on every rank
        assert n == 256
        assert digests[0] != digests[1]        # independent batches
        assert thr == world * 256 * 4 / 20e-3  # whole-job aggregate


def test_bench_gpus_flag_spawns_ranks():
    """`bench.py --gpus 2` outside torchrun re-launches itself with two ranks (the same path the CUDA
    arm takes); the reference arm runs here on CPU: rank 0 prints the one JSON line, rank 1 exits 0."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--impl", "reference",
                        "--small", "--config", "1", "--steps", "1", "--warmup", "0", "--cpu-seconds", "0.5"],
                       capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    rec = json.loads(lines[0])
    assert rec["impl"] == "reference" and rec["ranks"] == 2 and rec["value"] > 0
    assert "torch.distributed.run" in r.stderr and "--nproc-per-node 2" in r.stderr
    assert rec["config"]["workload"].startswith("configs[0]")

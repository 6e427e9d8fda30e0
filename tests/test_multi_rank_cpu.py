"""N > 1 path of bench.py on CPU (gloo, world_size 2): replicas only -- every rank searches its own
light curve of the same shape, there is no data-path collective, and the job time is the maximum over
ranks."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    w = bench.build_workload("c1", curve=rank)
    # same shape on every rank (weak scaling), different noise realisation
    shape = (w.lc.n, w.n_per, w.n_dur)
    shapes = [None] * world
    dist.all_gather_object(shapes, shape)
    sums = [None] * world
    dist.all_gather_object(sums, float(w.lc.y[:16].sum()))
    t = bench.max_over_ranks(10.0 + 5.0 * rank, world)          # slowest rank defines the step time
    dist.barrier()
    if rank == 0:
        out.put((shapes, sums, t, world * w.trials))
    dist.destroy_process_group()


def test_two_rank_replicas_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    shapes, sums, t, trials = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert shapes[0] == shapes[1]
    assert sums[0] != sums[1]
    assert t == 15.0
    assert trials == 2 * shapes[0][1] * shapes[0][2]


def test_max_over_ranks_single_process():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5

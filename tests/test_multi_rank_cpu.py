"""N > 1 path of bench.py on CPU (gloo, world_size 2): replicas only -- every rank searches its own
light curve of the same shape, there is no data-path collective, and the job time is the maximum over
ranks."""
import os
import sys

import numpy as np
import pytest
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


# ---- period-sharded search: the sharding / all-gather / merge plumbing on CPU ----
def _oracle_search_stub(t, y, dy, periods, durations, tmpl, *, dt0, sde_kernel, **kw):
    """Stands in for gtls_search (no GPU here): same result layout, computed by the oracle."""
    import oracle
    import paper_2607_00348_b200 as g
    o = oracle.search(t, y, dy, periods, durations, tmpl, dt0=dt0)
    best = np.zeros(len(periods), dtype=g.BEST_DTYPE)
    for k in ("dur_idx", "start", "depth", "t0"):
        best[k] = o.best[k]
    raw = best.view(np.uint8).reshape(len(periods), g.BEST_DTYPE.itemsize)
    return g.SearchResult(o.chi2, None, None, raw, {"windows_evaluated": o.windows, "chi2_null": o.chi2_null}, 0)


def _oracle_sde_stub(chi2, *, sde_kernel):
    import oracle
    s = oracle.sde(np.asarray(chi2), sde_kernel)
    summ = {"best_period_idx": s.best_period_idx, "sde_argmax": s.sde_argmax, "chi2_min": float(np.min(chi2)),
            "sde_max": float(s.sde[s.sde_argmax]), "sde_raw_max": float(s.sde_raw.max())}
    return s.sde_raw, s.sde, summ, 0


def _shard_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import gtls_inputs as gi
    import paper_2607_00348_b200 as g
    w = gi.make_workload(1).subset(29)                   # 106 periods: not a multiple of the world size
    r = g._sharded_search(_oracle_search_stub, _oracle_sde_stub, w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations,
                          w.tmpl, dt0=0.05, sde_kernel=31)
    out.put((rank, np.asarray(r.chi2), r.best().copy(), np.asarray(r.sde), r.summary))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_period_sharded_search_gloo(world):
    sys.path.insert(0, ROOT)
    import gtls_inputs as gi
    import oracle
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + (os.getpid() % 2000) + world
    procs = [ctx.Process(target=_shard_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = [q.get(timeout=240) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = gi.make_workload(1).subset(29)
    ref = oracle.search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, dt0=0.05)
    s = oracle.sde(ref.chi2, 31)
    for rank, chi2, best, sde, summ in got:
        assert np.array_equal(chi2, ref.chi2)                       # every rank holds the full spectrum, in grid order
        for k in ("dur_idx", "start", "depth", "t0"):
            assert np.array_equal(best[k], ref.best[k])
        assert np.array_equal(sde, s.sde)
        assert summ["best_period_idx"] == s.best_period_idx
        assert summ["best_period"] == w.periods[s.best_period_idx]
        assert summ["best_start"] == ref.best["start"][s.best_period_idx]
        assert summ["windows_evaluated"] == ref.windows

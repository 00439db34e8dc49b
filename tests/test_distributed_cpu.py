"""The N > 1 path of bench.py shards independent sources across ranks with no data-path collective
(SURVEY.md 8(e)); the only collectives are the barrier and the MAX over ranks of the step time.  This
world_size-2 gloo test covers that host logic: disjoint source indices per rank and the MAX reduction."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    cfg, hp, hc, ang, metas = bench.make_inputs("cfg1", rank)
    t = torch.tensor([10.0 + rank], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    gathered = [None] * world
    dist.all_gather_object(gathered, (float(hp[0, 100]), tuple(ang[0])))
    dist.barrier()
    if rank == 0:
        out.put((float(t.item()), gathered))
    dist.destroy_process_group()


def test_two_ranks_get_disjoint_sources_and_max_time():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, 29541, out)) for r in range(2)]
    for p in procs:
        p.start()
    tmax, gathered = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert tmax == 11.0
    assert gathered[0] != gathered[1]      # different seeds -> different sources per rank


# ---- one long series split in time over the ranks: no exchange step, each rank re-reads a halo ------------
def _time_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import numpy as np
    import workloads as W
    import paper_2505_09600_b200 as ltdi
    from oracle import Oracle
    orc = Oracle("f80", threads=2)
    cfg = W.config(2, n=9001)
    hp, hc, ang, _ = W.source(cfg, 0)
    gen, order, fd = 20, 31, 2
    pieces = {}
    for which in ("full", "lfa"):
        lo, hi = orc.margins(cfg["orbit"], gen, order, 0 if which == "full" else fd)
        sub, src, dst, a, b = ltdi.time_shard(cfg["orbit"], lo, hi, world, rank)
        if which == "full":
            r = orc.response_full(sub, hp[src], hc[src], ang, gen, order, want=())
        else:
            r = orc.response_lfa(sub, hp[src], hc[src], ang, gen, order, fd, want=())
        pieces[which] = (a, b, {c: r[c][0, dst] for c in "AET"})
    gathered = [None] * world
    dist.all_gather_object(gathered, pieces)
    if rank == 0:
        worst = 0.0
        for which in ("full", "lfa"):
            lo, hi = orc.margins(cfg["orbit"], gen, order, 0 if which == "full" else fd)
            ref = (orc.response_full(cfg["orbit"], hp, hc, ang, gen, order, want=()) if which == "full"
                   else orc.response_lfa(cfg["orbit"], hp, hc, ang, gen, order, fd, want=()))
            ends = sorted((g[which][0], g[which][1]) for g in gathered)
            assert ends[0][0] == lo and ends[-1][1] == cfg["n"] - hi
            assert all(ends[i][1] == ends[i + 1][0] for i in range(world - 1))     # contiguous, disjoint, complete
            for c in "AET":
                got = np.zeros(cfg["n"])
                for g in gathered:
                    a, b, r = g[which]
                    got[a:b] = r[c]
                scale = max(np.linalg.norm(ref[k][0]) for k in "AET")
                worst = max(worst, float(np.linalg.norm(got - ref[c][0]) / scale))
        out.put(worst)
    dist.barrier()
    dist.destroy_process_group()


def test_one_series_split_in_time_over_two_ranks():
    """the stitched pieces are the whole-series response (the sub-grids' t0 is rounded to fp64: 1e-15, not bitwise)"""
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_time_worker, args=(r, 2, 29543, out)) for r in range(2)]
    for p in procs:
        p.start()
    worst = out.get(timeout=300)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert worst < 1e-13, worst


def test_time_shard_arguments():
    sys.path.insert(0, ROOT)
    import pytest
    import workloads as W
    import paper_2505_09600_b200 as ltdi
    d = W.orbit_desc(1000, 5.0, t0=100.0)
    cover = []
    for r in range(3):
        sub, src, dst, a, b = ltdi.time_shard(d, 150, 120, 3, r)
        assert sub["n"] == src.stop - src.start == (b - a) + 270 and sub["t0"] == 100.0 + 5.0 * src.start
        assert dst == slice(150, 150 + b - a) and src.start == a - 150 and src.stop == b + 120
        cover.append((a, b))
    assert cover[0][0] == 150 and cover[-1][1] == 880 and all(cover[i][1] == cover[i + 1][0] for i in range(2))
    with pytest.raises(ValueError):
        ltdi.time_shard(d, 150, 120, 3, 3)
    with pytest.raises(ValueError):
        ltdi.time_shard(d, 600, 500, 2, 0)

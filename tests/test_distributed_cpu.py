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

"""N > 1 path of bench.py on CPU: world_size 2 over gloo.  The path shards over independent model
evaluations: every rank owns a disjoint range of model indices, there is no
data-path collective, and a job's time is the slowest rank's (all_reduce MAX)."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    batch = 3
    m0 = bench.shard_models(batch, rank)
    mine = list(range(m0, m0 + batch))
    gathered = [None] * world
    dist.all_gather_object(gathered, mine)
    t = bench.max_over_ranks(10.0 * (rank + 1))            # rank r "took" 10 (r + 1) ms
    rate = bench.whole_job_rate(batch * 5, world, t * 1e-3)
    if rank == 0:
        out.put((gathered, t, rate))
    dist.destroy_process_group()


def test_two_ranks_shard_models_and_take_the_slowest_time():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    gathered, t, rate = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    flat = [i for g in gathered for i in g]
    assert sorted(flat) == list(range(6)) and len(set(flat)) == 6     # disjoint, contiguous cover
    assert t == 20.0                                                   # max over ranks
    assert abs(rate - (3 * 5 * 2) / 0.020) < 1e-9                      # all ranks' units / slowest time


def test_single_rank_is_identity():
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.shard_models(4, 0) == 0 and bench.shard_models(4, 3) == 12

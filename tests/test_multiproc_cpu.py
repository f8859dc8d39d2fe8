"""World-size-2 gloo test (CPU) of the only N>1 host logic there is: replicas whose timings are combined
as max-over-ranks and whose unit counts are summed (the path does not shard)."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, launches = bench.combine_over_ranks(10.0 + 5.0 * rank, 100 + rank, torch.device("cpu"), world)
    q.put((rank, ms, launches))
    dist.destroy_process_group()


def test_replica_timing_is_max_over_ranks_and_launches_sum():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, 29613, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
    assert all(abs(ms - 15.0) < 1e-12 and n == 201 for _, ms, n in res)

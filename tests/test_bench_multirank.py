"""N > 1 host logic of bench.py ("replicas only") on CPU: two gloo ranks, the
max-over-ranks timing and the whole-job aggregate.  No GPU, no kernels."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = [3.0, 5.0][rank]                       # rank 1 is the slow one
    mx = bench.max_over_ranks(ms, world, "cpu")
    value = bench.aggregate([1000 * 10] * world, mx)
    out.put((rank, mx, value))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_max_and_aggregate():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mx, value in res:
        assert mx == 5.0                                        # max over ranks, not the own time
        assert abs(value - 2 * 1000 * 10 / 5e-3 / 1e6) < 1e-9   # all ranks' updates / slowest rank


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.max_over_ranks(2.5, 1) == 2.5
    assert abs(bench.aggregate([8 * 4], 2.0) - 32 / 2e-3 / 1e6) < 1e-12

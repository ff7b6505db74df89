"""CPU, world_size 2, gloo: the multi-GPU contract of bench.py is "replicas only":
rank timing is reduced with MAX over ranks and the job value counts every rank's bytes."""
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
    ms = bench.max_over_ranks(1.0 + rank * 0.5, world, "cpu")          # rank 1 is the slow replica
    val = bench.job_value(274.4e6, world, ms)
    dist.barrier()
    out.put((rank, ms, val))
    dist.destroy_process_group()


def test_max_over_ranks_and_job_value_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, val in res:
        assert ms == 1.5                                      # MAX over ranks, identical on every rank
        assert abs(val - 2 * 274.4e6 / 1.5e-3 / 1e9) < 1e-6   # both replicas' bytes / slowest time


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(2.25, 1, "cpu") == 2.25
    assert bench.job_value(1e9, 1, 1.0) == 1000.0

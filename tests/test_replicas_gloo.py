"""The N > 1 path of bench.py on CPU: world_size-2 gloo.  The hot path does not shard (north_star:
one GPU, no collectives; DESIGN.md section 9 "replicas only"), so the only multi-rank logic is the
aggregation of N independent replicas: job time = max over ranks, job work = sum over ranks."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 if rank == 0 else 12.5          # rank 1 is the slow replica
    value, ms = bench.job_value(ms_local, cells_per_rank=1000, steps=4, world=world, device="cpu")
    dist.barrier()
    if rank == 0:
        out.put((value, ms))
    dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_replica_aggregation_world_size_2():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    value, ms = out.get(timeout=90)
    for p in procs:
        p.join(timeout=30)
        assert p.exitcode == 0
    assert ms == 12.5                                 # max over ranks
    assert value == pytest.approx(2 * 1000 * 4 / 12.5e-3)   # both replicas' cells over the slowest time


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    value, ms = bench.job_value(5.0, 10, 2, 1)
    assert ms == 5.0 and value == pytest.approx(10 * 2 / 5e-3)

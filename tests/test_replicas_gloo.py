"""N > 1 runs N independent replicas (north_star fixes one GPU, no data-path collective).
The only distributed logic is bench.py's aggregation — time = MAX over ranks, work = SUM — covered here with
world_size 2 on the gloo backend (CPU)."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import bench

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms, iters, launches = bench.aggregate_over_ranks(100.0 + 50.0 * rank, 180 * (rank + 1), 900 + rank, dist, "cpu")
        dist.barrier()
        out.put((rank, ms, iters, launches))
    finally:
        dist.destroy_process_group()


def test_replica_aggregation_world_size_2():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, iters, launches in res:
        assert ms == 150.0                      # MAX over ranks
        assert iters == 180 + 360               # SUM: whole-job iterations
        assert launches == 900 + 901
    # the metric of the job: iterations of all replicas / slowest replica's time
    assert abs(res[0][2] / (res[0][1] * 1e-3) - 3600.0) < 1e-9


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.aggregate_over_ranks(12.5, 180, 905, None, "cpu") == (12.5, 180, 905)

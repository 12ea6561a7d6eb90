"""N>1 host logic on CPU (gloo, world_size 2): the path does not shard (replicas only), so the only
cross-rank step is the timing aggregation of bench.py — MAX of the times, SUM of the units."""
import os
import socket
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import bench
    r, w = bench.init_dist("gloo")
    assert (r, w) == (rank, world) and bench.dist_env() == (rank, world, rank)
    bench.barrier()
    ms, units = bench.aggregate_over_ranks(10.0 + 5.0 * rank, 100.0 * (rank + 1))
    q.put((rank, ms, units))
    bench.barrier()
    import torch.distributed as dist
    dist.destroy_process_group()


def test_aggregate_over_two_ranks():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(0, 15.0, 300.0), (1, 15.0, 300.0)]      # max over ranks, sum of units


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_over_ranks(3.5, 7.0) == (3.5, 7.0)
    assert abs(bench.FP32_PEAK_TFLOPS - 74.45) < 0.01

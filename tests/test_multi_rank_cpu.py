"""N > 1 path on the CPU (world_size 2, gloo): the path is "replicas only", so the only multi-rank
logic is bench.py's aggregation — max-over-ranks timing and the whole-job value.  No CUDA, no oracle."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = [10.0 + 5.0 * rank, 100.0 - 7.0 * rank]          # rank 1 is slower on [0], rank 0 on [1]
        red = bench.max_over_ranks(mine)
        dist.barrier()
        q.put((rank, red))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert out[0] == out[1] == [15.0, 100.0]


def test_whole_job_value_is_aggregate_over_replicas():
    sys.path.insert(0, ROOT)
    import bench
    one = bench.whole_job_value(1, 512 ** 3, 22, 0.05)
    assert one == pytest.approx(512 ** 3 * 22 / 0.05)
    assert bench.whole_job_value(8, 512 ** 3, 22, 0.05) == pytest.approx(8 * one)   # weak scaling: replicas add up
    assert bench.whole_job_value(1, 10, 0, 0.05) == 0.0
    assert bench.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]                            # no process group: identity

"""N > 1 path of bench.py on CPU: two gloo ranks agree on the max-over-ranks time and rank 0 forms the
whole-job rate of independent replicas (the path has no exchange step)."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        local_ms = 10.0 + 5.0 * rank            # rank 1 is the slow one
        dist.barrier()
        ms = bench.max_over_ranks(dist, local_ms, device="cpu")
        rate = bench.replicas_throughput(world, 360, ms * 1e-3)
        out.put((rank, ms, rate))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_two_gloo_ranks_max_time_and_replica_rate():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=100) for _ in ps)
    for p in ps:
        p.join(timeout=30)
        assert p.exitcode == 0
    for rank, ms, rate in res:
        assert ms == 15.0                               # every rank sees the slowest rank's time
        assert abs(rate - 2 * 360 / 0.015) < 1e-6       # two replicas, each the whole orbit


def test_single_process_is_identity():
    import bench
    assert bench.max_over_ranks(None, 3.5) == 3.5
    assert bench.replicas_throughput(1, 360, 0.072) == 360 / 0.072

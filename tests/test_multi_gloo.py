"""-m "not gpu": the N > 1 plumbing (replicas only) on two gloo processes:
host-side barrier group, max-over-ranks timing, whole-job aggregation."""
import os
import socket

import pytest


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q) -> None:
    import torch.distributed as dist

    from paper_2607_02630_b200 import multi

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        g = multi.host_group(dist)
        assert g is not None
        multi.host_barrier(dist, g)
        # rank r "measured" (10 + 5 r) ms for (r + 1) GB
        value, ms = multi.job_throughput(10.0 + 5.0 * rank, (rank + 1) * 10**9, dist, g)
        multi.host_barrier(dist, g)
        q.put((rank, value, ms))
    finally:
        dist.destroy_process_group()


def test_two_rank_aggregation():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    [p.start() for p in ps]
    out = sorted(q.get(timeout=120) for _ in ps)
    [p.join(60) for p in ps]
    assert all(p.exitcode == 0 for p in ps)
    for rank, value, ms in out:
        assert ms == pytest.approx(15.0)                      # the slowest rank
        assert value == pytest.approx(3e9 / 15e-3)            # all ranks' bytes over that time


def test_single_process_passthrough():
    from paper_2607_02630_b200 import multi

    value, ms = multi.job_throughput(4.0, 8 * 10**9)
    assert ms == 4.0 and value == pytest.approx(2e12)

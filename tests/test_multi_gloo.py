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


def test_bench_rank_logic_two_ranks_on_gloo():
    """bench.py's own N-rank logic, launched the way the driver launches it (torch.distributed.run, one rank per
    GPU), with the GPU work left out: rank 0 prints n_gpus == 2, the max over ranks and the summed bytes."""
    import json
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(root, "bench.py"), "--gpus", "2", "--plumbing-check"]
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=root)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [json.loads(ln) for ln in p.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, p.stdout
    d = lines[0]
    assert d["n_gpus"] == 2 and d["ms_max"] == pytest.approx(11.0) and d["value"] == pytest.approx(2.0 / 11e-3)


def test_bench_refuses_a_rank_count_that_is_not_gpus():
    """--gpus 4 under a 1-rank launch (or on a node with fewer GPUs) must fail loudly, not print n_gpus: 1."""
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0")
    p = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "4", "--plumbing-check"], capture_output=True,
                       text=True, timeout=120, cwd=root, env=env)
    assert p.returncode != 0 and "n_gpus would lie" in (p.stderr + p.stdout)
    import torch

    if torch.cuda.device_count() < 4:
        env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
        p = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "4", "--steps", "1"], capture_output=True,
                           text=True, timeout=120, cwd=root, env=env)
        assert p.returncode != 0 and "GPU(s)" in (p.stderr + p.stdout)

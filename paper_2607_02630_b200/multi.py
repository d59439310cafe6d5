"""Multi-GPU plumbing: replicas only.

Requests are independent and CTR blocks inside a request are independent, so the path shards with no
exchange step: one process per GPU, each with its own engine (ring + persistent kernel + mailbox),
no data-path collective, NVLink unused.  What the ranks do share is bookkeeping, and that is all this
module holds: lining up before a timed region without launching a kernel (the persistent engine owns
every SM's shared memory, so a NCCL barrier kernel could wait for it forever) and reducing the
per-rank device times to the job's figure (max over ranks).  No cipher arithmetic here.
"""
from __future__ import annotations


def host_group(dist):
    """A gloo group over all ranks for host-side barriers while the engine runs (None if single process)."""
    if not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return None
    return dist.new_group(backend="gloo")


def host_barrier(dist, group) -> None:
    if group is not None:
        dist.barrier(group=group)


def job_throughput(ms_local: float, bytes_local: int, dist=None, group=None):
    """(whole-job bytes per second, max-over-ranks milliseconds): every rank processed bytes_local in
    ms_local of device time; the job took as long as its slowest rank."""
    import torch

    ms_max, total = float(ms_local), int(bytes_local)
    if dist is not None and dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        t = torch.tensor([float(ms_local)], dtype=torch.float64)
        b = torch.tensor([int(bytes_local)], dtype=torch.int64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
        dist.all_reduce(b, op=dist.ReduceOp.SUM, group=group)
        ms_max, total = float(t.item()), int(b.item())
    return total / (ms_max * 1e-3), ms_max

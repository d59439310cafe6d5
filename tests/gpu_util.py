"""Helpers shared by the -m gpu tests: device buffers through torch (plumbing only), the oracle
run over many requests on a thread pool, and an engine fixture with a safety idle-exit."""
from __future__ import annotations

import concurrent.futures as cf
import os

import numpy as np

from oracle import oracle as o


def torch_cuda():
    import torch

    if not torch.cuda.is_available():
        raise RuntimeError("this test needs a CUDA device")
    return torch


def to_device(arr: np.ndarray):
    """uint8 numpy -> uint8 CUDA tensor (16-byte aligned by the caching allocator)."""
    torch = torch_cuda()
    t = torch.from_numpy(np.array(arr)).to("cuda:0", non_blocking=False)  # a writable copy
    assert t.data_ptr() % 16 == 0
    return t


def device_empty(n: int):
    torch = torch_cuda()
    return torch.empty(max(int(n), 1), dtype=torch.uint8, device="cuda:0")


def stream_sync():
    """Synchronise torch's current stream only (a device-wide sync would block on the engine)."""
    torch_cuda().cuda.current_stream().synchronize()


def oracle_many(jobs, workers: int | None = None):
    """jobs: list of (key, icb, data, block_offset) -> list of bytes, on a thread pool
    (the ctypes call into the C oracle releases the GIL)."""
    workers = workers or max(1, len(os.sched_getaffinity(0)))
    with cf.ThreadPoolExecutor(workers) as ex:
        return list(ex.map(lambda j: o.ctr(j[0], j[1], j[2], j[3] if len(j) > 3 else 0), jobs))


def first_mismatch(got: np.ndarray, want: bytes) -> int:
    w = np.frombuffer(want, dtype=np.uint8)
    if got.shape != w.shape:
        return -2
    ne = np.nonzero(got != w)[0]
    return int(ne[0]) if ne.size else -1


def verify_requests(w, idxs, out_of, workers: int | None = None):
    """Every byte of requests `idxs` of workload `w` against the oracle, on a thread pool (the payload is
    regenerated from the seed, the oracle call releases the GIL).  out_of(i) -> uint8 ndarray of request i's
    output.  Returns [(request, first mismatching byte or -2 for a length mismatch)], empty when all match."""
    workers = workers or max(1, len(os.sched_getaffinity(0)))

    def one(i):
        want = o.ctr(w.key_of(i), w.icb_of(i), w.payload(i))
        return i, first_mismatch(out_of(i), want)

    with cf.ThreadPoolExecutor(workers) as ex:
        return [(i, b) for i, b in ex.map(one, idxs) if b != -1]

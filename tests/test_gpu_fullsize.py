"""-m gpu parity at BASELINE.json's FULL config sizes, in the launch configuration bench.py times (the native
closed loop `aes_loop_run` on the persistent engine, the config's own window), every byte against the oracle:

    configs[1]  1,000 x 1 MiB  AES-128, one key, 64 in flight                      1.05 GB
    configs[2]    200 x 8 MiB  AES-256, one key, 16 in flight                      1.68 GB
    configs[3] 10,000 requests 1-64 KiB + tails, per-request AES-128/256 keys      0.16 GB
               (key expansion on the path), fully random ICBs, 256 in flight; also from 4 executor threads

SURVEY.md section 8(d) "Parity coverage": the oracle on every byte of C1-C4 (configs[0] is in test_gpu_engine.py).
The oracle runs on all host cores beside the check (0.3-0.45 GB/s on 16 cores: a few seconds per config).
"""
import numpy as np
import pytest

from paper_2607_02630_b200 import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def E():
    import paper_2607_02630_b200.binding as B
    import gpu_util as G

    torch = G.torch_cuda()
    torch.zeros(1, device="cuda:0")
    torch.cuda.synchronize()
    B.aes_engine_start(0, idle_exit_ms=120000)
    yield B
    B.aes_engine_stop()


def _fixed_size_config(E, w, threads=1):
    """Runs all of w (equal-sized requests, one key) through the closed loop and checks every byte."""
    import gpu_util as G

    torch = G.torch_cuda()
    n, size = w.n, int(w.length[0])
    src = torch.empty(n * size, dtype=torch.uint8, device="cuda:0")
    dst = torch.empty(n * size, dtype=torch.uint8, device="cuda:0")
    stage = torch.empty(size, dtype=torch.uint8).pin_memory()
    for i in range(n):
        stage.numpy()[:] = w.payload(i)
        src[i * size:(i + 1) * size].copy_(stage)   # H2D memcpy, no kernel (the engine owns the SMs)
        G.stream_sync()
    marker = torch.full((size,), 0xA5, dtype=torch.uint8).pin_memory()
    for i in range(n):
        dst[i * size:(i + 1) * size].copy_(marker, non_blocking=True)  # a request that never ran is not "right by chance"
    G.stream_sync()
    srcs = np.asarray([src.data_ptr() + i * size for i in range(n)], dtype=np.uint64)
    dsts = np.asarray([dst.data_ptr() + i * size for i in range(n)], dtype=np.uint64)
    ctx = E.aes_ctx_create(w.key_of(0))
    r = E.aes_loop_run(w.icb, srcs, dsts, w.length, window=w.in_flight, ctx=ctx, threads=threads)
    E.aes_ctx_destroy(ctx)
    assert r["requests"] == n and r["bytes"] == w.total_bytes
    assert r["max_in_flight"] <= w.in_flight
    out = dst.cpu().numpy()
    bad = G.verify_requests(w, range(n), lambda i: out[i * size:(i + 1) * size])
    assert not bad, "first mismatches (request, byte): %s" % bad[:5]
    return n * size


def test_config2_full_every_byte(E):
    """configs[1]: 1,000 x 1 MiB AES-128-CTR, 64 in flight -- the bench workload, every byte."""
    assert _fixed_size_config(E, workloads.config2()) == 1000 << 20


def test_config3_full_every_byte(E):
    """configs[2]: 200 x 8 MiB AES-256-CTR, 16 in flight, every byte."""
    assert _fixed_size_config(E, workloads.config3()) == 200 * (8 << 20)


@pytest.mark.parametrize("threads", [1, 4])
def test_config4_full_every_byte(E, threads):
    """configs[3]: all 10,000 requests of the fine-grained mix, per-request keys expanded on the device, 256 in
    flight, from one executor thread and from four; every byte."""
    import gpu_util as G

    torch = G.torch_cuda()
    w = workloads.config4()
    assert w.n == 10000
    stride = 64 * 1024 + 16
    src = torch.empty(w.n * stride, dtype=torch.uint8, device="cuda:0")
    dst = torch.empty(w.n * stride, dtype=torch.uint8, device="cuda:0")
    host = np.full(w.n * stride, 0x5A, dtype=np.uint8)
    for i in range(w.n):
        host[i * stride:i * stride + int(w.length[i])] = w.payload(i)
    src.copy_(torch.from_numpy(host))
    dst.copy_(torch.from_numpy(np.full(w.n * stride, 0xA5, dtype=np.uint8)))
    G.stream_sync()
    keys = np.zeros((w.n, 32), dtype=np.uint8)
    keybits = np.zeros(w.n, dtype=np.int32)
    for i in range(w.n):
        k = w.key_of(i)
        keys[i, :len(k)] = np.frombuffer(k, dtype=np.uint8)
        keybits[i] = 8 * len(k)
    srcs = np.asarray([src.data_ptr() + i * stride for i in range(w.n)], dtype=np.uint64)
    dsts = np.asarray([dst.data_ptr() + i * stride for i in range(w.n)], dtype=np.uint64)
    r = E.aes_loop_run(w.icb, srcs, dsts, w.length, window=w.in_flight, keys=keys, keybits=keybits, threads=threads)
    assert r["requests"] == w.n and r["bytes"] == w.total_bytes
    out = dst.cpu().numpy()
    bad = G.verify_requests(w, range(w.n), lambda i: out[i * stride:i * stride + int(w.length[i])])
    assert not bad, "first mismatches (request, byte): %s" % bad[:5]
    # nothing written past the end of any request (the 16 spare bytes still hold the marker)
    tails = np.concatenate([out[i * stride + int(w.length[i]):(i + 1) * stride] for i in range(0, w.n, 7)])
    assert (tails == 0xA5).all()

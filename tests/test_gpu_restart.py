"""-m gpu: engine life cycle across aes_engine_stop / aes_engine_start (own module: the engine tests
keep one engine running for the whole module)."""
import numpy as np
import pytest

from paper_2607_02630_b200 import workloads

pytestmark = pytest.mark.gpu


def test_installed_context_survives_restart():
    """A context whose key sits in the key table keeps working across aes_engine_stop/start, with the
    same ring geometry (table kept) and with another one (table rebuilt, the key is installed again)."""
    import gpu_util as G
    import paper_2607_02630_b200.binding as B
    from oracle import oracle as o

    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7700]))
    key = rng.bytes(32)
    data = np.frombuffer(rng.bytes(20000), dtype=np.uint8)
    src = G.to_device(data)
    dst = G.device_empty(len(data))
    G.stream_sync()
    ctx = B.aes_ctx_create(key)
    for ring_slots in (0, 0, 256, 0):
        B.aes_engine_start(0, ring_slots=ring_slots, idle_exit_ms=60000)
        try:
            for _ in range(4):
                icb = rng.bytes(16)
                B.aes_wait(B.aes_ctr_submit(ctx, icb, src.data_ptr(), dst.data_ptr(), len(data)))
                assert dst.cpu().numpy().tobytes() == o.ctr(key, icb, data)
        finally:
            B.aes_engine_stop()
    B.aes_ctx_destroy(ctx)


def test_half_installed_context_starts_over_after_a_rebuilt_key_table():
    """A context used exactly twice has asked for its key to be filed (INSTALLING) and nobody has looked at that
    request's completion yet.  When the key table is rebuilt in that state (another ring size), the next submit must
    file the key again and the one after it must find it INSTALLED -- not ship the raw key with every request for ever."""
    import ctypes

    import gpu_util as G
    import paper_2607_02630_b200.binding as B
    from oracle import oracle as o

    state = B._lib.aesoff_test_ctx_state
    state.restype, state.argtypes = ctypes.c_int, [ctypes.c_void_p, ctypes.c_int]
    INSTALLING, INSTALLED = 2, 3
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7705]))
    key = rng.bytes(24)
    data = np.frombuffer(rng.bytes(9000), dtype=np.uint8)
    src, dst = G.to_device(data), G.device_empty(len(data))
    G.stream_sync()
    ctx = B.aes_ctx_create(key)

    def once():
        icb = rng.bytes(16)
        B.aes_wait(B.aes_ctr_submit(ctx, icb, src.data_ptr(), dst.data_ptr(), len(data)))
        assert dst.cpu().numpy().tobytes() == o.ctr(key, icb, data)

    B.aes_engine_start(0, ring_slots=512, idle_exit_ms=60000)
    try:
        once()
        once()
        assert state(ctx, 0) == INSTALLING
    finally:
        B.aes_engine_stop()
    B.aes_engine_start(0, ring_slots=128, idle_exit_ms=60000)  # other geometry: the key table is rebuilt
    try:
        once()
        assert state(ctx, 0) == INSTALLING  # filed again, under the new table
        once()
        assert state(ctx, 0) == INSTALLED
        once()
    finally:
        B.aes_engine_stop()
    B.aes_ctx_destroy(ctx)


def test_idle_exit_is_detected_and_engine_restarts():
    """Failure detection: a persistent kernel that has exited -- here by its own idle
    timer -- is seen through the host-mapped alive word: submits fail with AES_E_STOPPED instead of hanging,
    aes_engine_stop still returns, and a fresh start serves requests again."""
    import time

    import gpu_util as G
    import paper_2607_02630_b200.binding as B
    from oracle import oracle as o

    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7710]))
    key, icb = rng.bytes(16), rng.bytes(16)
    data = np.frombuffer(rng.bytes(5000), dtype=np.uint8)
    src, dst = G.to_device(data), G.device_empty(len(data))
    G.stream_sync()
    ctx = B.aes_ctx_create(key)
    B.aes_engine_start(0, idle_exit_ms=50)
    try:
        B.aes_wait(B.aes_ctr_submit(ctx, icb, src.data_ptr(), dst.data_ptr(), len(data)))
        assert B.aes_engine_info()["running"] == 1
        deadline = time.time() + 5.0
        while B.aes_engine_info()["running"] == 1 and time.time() < deadline:
            time.sleep(0.02)
        assert B.aes_engine_info()["running"] == 0, "the kernel should have left after 50 ms without requests"
        with pytest.raises(B.AesOffError) as e:
            B.aes_ctr_submit(ctx, icb, src.data_ptr(), dst.data_ptr(), len(data))
        assert e.value.code == B.AES_E_STOPPED
    finally:
        B.aes_engine_stop()
    B.aes_engine_start(0, idle_exit_ms=60000)
    try:
        dst = G.to_device(np.zeros(len(data), dtype=np.uint8))  # a copy, not a kernel: the engine owns the SMs
        G.stream_sync()
        B.aes_wait(B.aes_ctr_submit(ctx, icb, src.data_ptr(), dst.data_ptr(), len(data)))
        assert dst.cpu().numpy().tobytes() == o.ctr(key, icb, data)
    finally:
        B.aes_engine_stop()
    B.aes_ctx_destroy(ctx)


def test_wait_timeout_then_completion():
    """aes_wait with a 1 ns budget on a 256 MiB request times out (AES_E_TIMEOUT) without disturbing the request;
    a later wait sees it complete, bit-exact on sampled windows."""
    import gpu_util as G
    import paper_2607_02630_b200.binding as B
    from oracle import oracle as o

    torch = G.torch_cuda()
    n = 256 << 20
    big = torch.zeros(n, dtype=torch.uint8, device="cuda:0")
    out = torch.empty_like(big)
    torch.cuda.synchronize()
    key, icb = bytes(range(32)), bytes(range(16))
    ctx = B.aes_ctx_create(key)
    B.aes_engine_start(0, idle_exit_ms=60000)
    try:
        h = B.aes_ctr_submit(ctx, icb, big.data_ptr(), out.data_ptr(), n)
        with pytest.raises(B.AesOffError) as e:
            B.aes_wait(h, 1)
        assert e.value.code == B.AES_E_TIMEOUT
        B.aes_wait(h, 20_000_000_000)
        assert B.aes_poll(h) is True
        zeros = np.zeros(4096, dtype=np.uint8)
        for off in (0, 4096 * 12345, n - 4096):
            assert out[off:off + 4096].cpu().numpy().tobytes() == o.ctr(key, icb, zeros, off // 16)
    finally:
        B.aes_engine_stop()
    B.aes_ctx_destroy(ctx)


def test_other_kernels_run_beside_the_engine():
    """A kernel of the process's own (a torch fill, launched once before so that CUDA has its module loaded)
    completes while the full-size engine is running, and the engine still computes bit-exact."""
    import time

    import gpu_util as G
    import paper_2607_02630_b200.binding as B
    from oracle import oracle as o

    torch = G.torch_cuda()
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7720]))
    key, icb = rng.bytes(16), rng.bytes(16)
    data = np.frombuffer(rng.bytes(300000 + 9), dtype=np.uint8)
    src, dst = G.to_device(data), G.device_empty(len(data))
    other = torch.empty(1 << 20, dtype=torch.uint8, device="cuda:0")
    other.fill_(1)               # first launch: lazy module loading happens here, not beside the engine
    torch.cuda.synchronize()
    ctx = B.aes_ctx_create(key)
    B.aes_engine_start(0, idle_exit_ms=20000)
    try:
        t0 = time.time()
        other.fill_(7)           # a kernel on torch's stream, beside 148 persistent CTAs
        G.stream_sync()
        assert time.time() - t0 < 5.0, "the fill had to wait for the engine"
        B.aes_wait(B.aes_ctr_submit(ctx, icb, src.data_ptr(), dst.data_ptr(), len(data)))
        assert dst.cpu().numpy().tobytes() == o.ctr(key, icb, data)
        assert int(other[12345:12346].cpu().numpy()[0]) == 7
    finally:
        B.aes_engine_stop()
    B.aes_ctx_destroy(ctx)


def test_engine_without_the_decryption_table():
    """AES_ENGINE_NO_DECRYPT: 200 KiB of shared memory per CTA instead of 223; CTR and ECB-encrypt work, the
    decrypting calls are refused."""
    import gpu_util as G
    import paper_2607_02630_b200.binding as B
    from oracle import oracle as o

    torch = G.torch_cuda()
    torch.zeros(1, device="cuda:0")
    torch.cuda.synchronize()
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 8500]))
    key, iv = rng.bytes(24), rng.bytes(16)
    data = np.frombuffer(rng.bytes(80000), dtype=np.uint8)
    s, d = G.to_device(data), G.device_empty(len(data))
    G.stream_sync()
    ctx = B.aes_ctx_create(key)
    B.aes_engine_start(0, idle_exit_ms=20000, flags=B.AES_ENGINE_NO_DECRYPT)
    try:
        assert B.aes_engine_info()["smem_bytes_per_cta"] == 200 * 1024
        B.aes_wait(B.aes_ctr_submit(ctx, iv, s.data_ptr(), d.data_ptr(), len(data)))
        assert d.cpu().numpy().tobytes() == o.ctr(key, iv, data)
        B.aes_wait(B.aes_ecb_submit(ctx, False, s.data_ptr(), d.data_ptr(), len(data)))
        assert d.cpu().numpy().tobytes() == o.ecb_encrypt(key, data)
        for call in (lambda: B.aes_ecb_submit(ctx, True, s.data_ptr(), d.data_ptr(), len(data)),
                     lambda: B.aes_cbc_decrypt_submit(ctx, iv, s.data_ptr(), d.data_ptr(), len(data))):
            with pytest.raises(B.AesOffError) as e:
                call()
            assert e.value.code == B.AES_E_INVAL
    finally:
        B.aes_engine_stop()
    B.aes_engine_start(0, idle_exit_ms=20000)
    try:
        assert B.aes_engine_info()["smem_bytes_per_cta"] == 223 * 1024
        B.aes_wait(B.aes_cbc_decrypt_submit(ctx, iv, s.data_ptr(), d.data_ptr(), len(data)))
        assert d.cpu().numpy().tobytes() == o.cbc_decrypt(key, iv, data)
    finally:
        B.aes_engine_stop()
    B.aes_ctx_destroy(ctx)


def test_ordinary_host_memory_after_registration():
    """The paper's buffer is the server's own memory (j.buf): a numpy array from the ordinary heap is
    page-locked in place with aes_host_register and submitted at its own address, in place and out of place."""
    import gpu_util as G
    import paper_2607_02630_b200.binding as B
    from oracle import oracle as o

    torch = G.torch_cuda()
    torch.zeros(1, device="cuda:0")
    torch.cuda.synchronize()
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 8600]))
    n = (1 << 20) + 4096 + 7
    pool = np.zeros(3 * (1 << 21), dtype=np.uint8)             # the "server's" buffer pool, registered once
    base = (pool.ctypes.data + 63) & ~63
    B.aes_host_register(pool.ctypes.data, pool.nbytes)
    with pytest.raises(B.AesOffError):
        B.aes_host_register(pool.ctypes.data, pool.nbytes)      # twice is an error, not a crash
    off = base - pool.ctypes.data
    src, dst = pool[off:off + n], pool[off + (1 << 21):off + (1 << 21) + n]
    src[:] = np.frombuffer(rng.bytes(n), dtype=np.uint8)
    plain = src.copy()
    key, icb = rng.bytes(32), rng.bytes(16)
    ctx = B.aes_ctx_create(key)
    B.aes_engine_start(0, idle_exit_ms=20000)
    try:
        B.aes_wait(B.aes_ctr_submit(ctx, icb, src.ctypes.data, dst.ctypes.data, n))
        assert dst.tobytes() == o.ctr(key, icb, plain)
        B.aes_wait(B.aes_ctr_submit(ctx, icb, src.ctypes.data, src.ctypes.data, n))   # in place, as accel_encrypt(j.buf, j.len)
        assert src.tobytes() == o.ctr(key, icb, plain)
        dev = G.device_empty(n)                                                      # host -> device as well
        B.aes_wait(B.aes_ctr_submit(ctx, icb, src.ctypes.data, dev.data_ptr(), n))
        assert dev.cpu().numpy()[:n].tobytes() == plain.tobytes()
    finally:
        B.aes_engine_stop()
    B.aes_host_unregister(pool.ctypes.data)
    B.aes_ctx_destroy(ctx)

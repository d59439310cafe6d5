"""-m gpu: the dispatcher warps (step a3).  Consecutive batches of 32 sequence numbers go round n_dispatchers
warps, tickets stay numbered in sequence order through the token the warps pass along, keys that arrive raw
are expanded by whichever warp takes the request.  Every byte against the oracle, for 1, 3 and 8 dispatchers,
on a small ring (256 slots, so batches wrap around it), from four executor threads whose slot writes
interleave (holes in the ready prefix), with per-request keys and with a shared context whose key moves
into the key table while requests of it are in flight."""
import numpy as np
import pytest

from paper_2607_02630_b200 import workloads

pytestmark = pytest.mark.gpu


def _mixed(rng, n):
    lens = [int(x) for x in rng.choice([0, 1, 16, 100, 4096, 4097, 20000, 65536, 65536 + 5, 300000], size=n)]
    datas = [np.frombuffer(rng.bytes(m), dtype=np.uint8) for m in lens]
    icbs = rng.integers(0, 256, size=(n, 16), dtype=np.uint8)
    return lens, datas, icbs


@pytest.mark.parametrize("n_disp", [1, 3, 8])
def test_parity_with_n_dispatchers(n_disp):
    import gpu_util as G
    import paper_2607_02630_b200.binding as B

    torch = G.torch_cuda()
    torch.zeros(1, device="cuda:0")
    torch.cuda.synchronize()
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 8100 + n_disp]))
    n = 1200
    lens, datas, icbs = _mixed(rng, n)
    stride = 300000 + 16
    host = np.full(n * stride, 0x5A, dtype=np.uint8)
    for i, d in enumerate(datas):
        host[i * stride:i * stride + len(d)] = d
    src = torch.empty(n * stride, dtype=torch.uint8, device="cuda:0")
    dst = torch.empty(n * stride, dtype=torch.uint8, device="cuda:0")
    src.copy_(torch.from_numpy(host))
    dst.copy_(torch.from_numpy(np.full(n * stride, 0xA5, dtype=np.uint8)))
    torch.cuda.synchronize()
    srcs = np.asarray([src.data_ptr() + i * stride for i in range(n)], dtype=np.uint64)
    dsts = np.asarray([dst.data_ptr() + i * stride for i in range(n)], dtype=np.uint64)
    keys = np.zeros((n, 32), dtype=np.uint8)
    keybits = np.zeros(n, dtype=np.int32)
    raw_keys = []
    for i in range(n):
        k = rng.bytes((16, 24, 32)[i % 3])
        raw_keys.append(k)
        keys[i, :len(k)] = np.frombuffer(k, dtype=np.uint8)
        keybits[i] = 8 * len(k)
    shared_key = rng.bytes(32)
    B.aes_engine_start(0, ring_slots=256, idle_exit_ms=60000, n_dispatchers=n_disp)
    try:
        info = B.aes_engine_info()
        assert info["n_dispatchers"] == n_disp and info["ring_slots"] == 256
        # (a) per-request keys (raw in every descriptor), four executor threads
        r = B.aes_loop_run(icbs, srcs, dsts, lens, window=200, keys=keys, keybits=keybits, threads=4)
        assert r["requests"] == n
        out = dst.cpu().numpy()
        wants = G.oracle_many([(raw_keys[i], icbs[i].tobytes(), datas[i]) for i in range(n)])
        for i in range(n):
            assert G.first_mismatch(out[i * stride:i * stride + lens[i]], wants[i]) == -1, "per-request key, request %d" % i
        tails = np.concatenate([out[i * stride + lens[i]:(i + 1) * stride][:64] for i in range(n)])
        assert (tails == 0xA5).all(), "bytes written past the end of a request"
        # (b) one shared context, window deeper than the ring is not allowed to matter: raw, then raw + install,
        #     then raw again until that request has completed, then by key-table index -- all in flight together
        dst.copy_(torch.from_numpy(np.full(n * stride, 0xA5, dtype=np.uint8)))
        G.stream_sync()
        ctx = B.aes_ctx_create(shared_key)
        r = B.aes_loop_run(icbs, srcs, dsts, lens, window=256, ctx=ctx, threads=2)
        assert r["requests"] == n
        B.aes_ctx_destroy(ctx)
        out = dst.cpu().numpy()
        wants = G.oracle_many([(shared_key, icbs[i].tobytes(), datas[i]) for i in range(n)])
        for i in range(n):
            assert G.first_mismatch(out[i * stride:i * stride + lens[i]], wants[i]) == -1, "shared context, request %d" % i
        info = B.aes_engine_info()
        assert info["cut_eighths"] + info["cut_halves"] + info["cut_rows"] >= 1
    finally:
        B.aes_engine_stop()


def test_idle_exit_with_several_dispatchers_and_restart():
    """The idle timer is dispatcher 0's; the others leave on its word.  Then a restart with another count."""
    import time

    import gpu_util as G
    import paper_2607_02630_b200.binding as B
    from oracle import oracle as o

    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 8150]))
    key = rng.bytes(16)
    data = np.frombuffer(rng.bytes(70000), dtype=np.uint8)
    src, dst = G.to_device(data), G.device_empty(len(data))
    G.stream_sync()
    ctx = B.aes_ctx_create(key)
    B.aes_engine_start(0, idle_exit_ms=50, n_dispatchers=4)
    try:
        for _ in range(40):  # more than one batch: the token has moved on from dispatcher 0
            icb = rng.bytes(16)
            B.aes_wait(B.aes_ctr_submit(ctx, icb, src.data_ptr(), dst.data_ptr(), len(data)))
        assert dst.cpu().numpy().tobytes() == o.ctr(key, icb, data)
        deadline = time.time() + 5.0
        while B.aes_engine_info()["running"] == 1 and time.time() < deadline:
            time.sleep(0.02)
        assert B.aes_engine_info()["running"] == 0
    finally:
        try:
            B.aes_engine_stop()
        except B.AesOffError:
            pass
    B.aes_engine_start(0, idle_exit_ms=60000, n_dispatchers=2)
    try:
        icb = rng.bytes(16)
        B.aes_wait(B.aes_ctr_submit(ctx, icb, src.data_ptr(), dst.data_ptr(), len(data)))
        assert dst.cpu().numpy().tobytes() == o.ctr(key, icb, data)
    finally:
        B.aes_engine_stop()
    B.aes_ctx_destroy(ctx)

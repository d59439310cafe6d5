"""-m gpu parity and behaviour of the persistent engine: submission ring -> dispatcher warp ->
service warps -> worker warps -> completion mailbox (steps a2, a3, a7 of SURVEY.md section 8(a)), against the
oracle, byte for byte.

While the engine runs, a device-wide synchronisation would block on the persistent kernel, so these
tests only use host<->device copies (no torch kernels) and stream-level synchronisation.
"""
import threading

import numpy as np
import pytest

from paper_2607_02630_b200 import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", params=["latency_units", "row_units_only"])
def P(request):
    """Every test runs twice: with the default unit policy (requests up to 64 KiB, and larger ones
    that find the GPU idle, are cut into 1/8-row units) and with whole-row units only."""
    import paper_2607_02630_b200.binding as B
    import gpu_util as G

    torch = G.torch_cuda()
    torch.zeros(1, device="cuda:0")  # CUDA context + torch's first kernels before the engine occupies the SMs
    torch.cuda.synchronize()
    B.aes_engine_start(0, idle_exit_ms=60000,
                       fine_rows=0 if request.param == "latency_units" else B.AES_FINE_ROWS_OFF)
    B.test_latency_units = request.param == "latency_units"
    yield B
    B.aes_engine_stop()


def _submit_all(P, reqs, in_place=False, host=False):
    """reqs: (key, icb, ndarray).  Submits everything (spinning on ring-full), waits, returns outputs."""
    import gpu_util as G

    ctxs, srcs, dsts, hs = {}, [], [], []
    for key, icb, data in reqs:
        if key not in ctxs:
            ctxs[key] = P.aes_ctx_create(key)
        s = G.to_device(data) if len(data) else G.device_empty(0)
        srcs.append(s)
        dsts.append(s if in_place else G.device_empty(len(data)))
    G.stream_sync()
    for (key, icb, data), s, d in zip(reqs, srcs, dsts):
        while True:
            try:
                hs.append(P.aes_ctr_submit(ctxs[key], icb, s.data_ptr(), d.data_ptr(), len(data)))
                break
            except P.AesOffError as e:
                if e.code != P.AES_E_AGAIN:
                    raise
    for h in hs:
        P.aes_wait(h, 20_000_000_000)
        assert P.aes_poll(h) is True
    outs = [d.cpu().numpy()[: len(x)] for d, (_, _, x) in zip(dsts, reqs)]
    for c in ctxs.values():
        P.aes_ctx_destroy(c)
    return outs


def _check(P, reqs, **kw):
    import gpu_util as G

    outs = _submit_all(P, reqs, **kw)
    wants = G.oracle_many([(k, i, d) for k, i, d in reqs])
    for n, (got, want) in enumerate(zip(outs, wants)):
        bad = G.first_mismatch(got, want)
        assert bad == -1, "request %d (len %d, keybits %d, icb %s): first mismatch at byte %d" % (
            n, len(reqs[n][2]), 8 * len(reqs[n][0]), reqs[n][1].hex(), bad)


def test_engine_info(P):
    info = P.aes_engine_info()
    assert info["running"] == 1 and info["n_ctas"] == info["sm_count"] >= 100
    assert info["kernel_launches"] >= 1


def test_config1_single_request(P):
    w = workloads.config1()
    _check(P, [(w.key_of(0), w.icb_of(0), w.payload(0))])


def test_lengths_and_carries(P):
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7000]))
    reqs = []
    for keylen in (16, 24, 32):
        key = rng.bytes(keylen)
        for n in (0, 1, 15, 16, 17, 4095, 4096, 4097, 16385, 65536 + 5, (1 << 20) + 5):
            reqs.append((key, rng.bytes(8) + bytes(8), np.frombuffer(rng.bytes(n), dtype=np.uint8)))
        for icb in workloads.edge_icbs():
            reqs.append((key, icb, np.frombuffer(rng.bytes(16 * 600 + 3), dtype=np.uint8)))
    _check(P, reqs)


def test_lone_requests_one_chunk_per_cta(P):
    """A lone request of more than one row per CTA is cut into ceil(rows / CTAs)-row chunks (not a power of
    two: 3 MiB -> 6 rows, 5 MiB + 5 -> 9, 7 MiB - 16 -> 13, 9 MiB -> 16), a counter that carries out of bytes
    14 and 13 inside it included.  One at a time, so that each finds the GPU idle; every byte checked."""
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7100]))
    info = P.aes_engine_info()
    icbs = [rng.bytes(8) + bytes(8), rng.bytes(12) + bytes([0x00, 0x00, 0xff, 0xf0]), rng.bytes(13) + bytes([0xff, 0xfe, 0x07])]
    for j, n in enumerate(((3 << 20), (5 << 20) + 5, (7 << 20) - 16, 9 << 20, 577 * 4096 + 1)):
        key = rng.bytes((16, 24, 32)[j % 3])
        data = np.frombuffer(rng.bytes(n), dtype=np.uint8)
        _check(P, [(key, icbs[j % 3], data)])
    after = P.aes_engine_info()
    assert after["running"] == 1 and after["kernel_launches"] == info["kernel_launches"]


def test_config2_shape_64_in_flight(P):
    """configs[1] at reduced count: 64 x 1 MiB AES-128, one key, distinct nonces, all 64 in flight."""
    w = workloads.config2(n=64)
    _check(P, [(w.key_of(i), w.icb_of(i), w.payload(i)) for i in range(w.n)])


def test_config3_shape_sampled(P):
    """configs[2] at reduced count: 16 x 8 MiB AES-256 in flight; sampled 64 KiB windows per request
    (first, last, 2 random) through oracle_ctr_at."""
    import gpu_util as G

    w = workloads.config3(n=16)
    ctx = P.aes_ctx_create(w.key_of(0))
    srcs = [G.to_device(w.payload(i)) for i in range(w.n)]
    dsts = [G.device_empty(int(w.length[i])) for i in range(w.n)]
    G.stream_sync()
    hs = [P.aes_ctr_submit(ctx, w.icb_of(i), srcs[i].data_ptr(), dsts[i].data_ptr(), int(w.length[i]))
          for i in range(w.n)]
    for h in hs:
        P.aes_wait(h, 20_000_000_000)
    P.aes_ctx_destroy(ctx)
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7100]))
    W = 64 << 10
    jobs, gots, tags = [], [], []
    for i in range(w.n):
        n = int(w.length[i])
        src_h = w.payload(i)
        out_h = dsts[i].cpu().numpy()
        for s0 in [0, n - W] + [int(x) * 16 for x in rng.integers(0, (n - W) // 16, size=2)]:
            jobs.append((w.key_of(i), w.icb_of(i), src_h[s0:s0 + W], s0 // 16))
            gots.append(out_h[s0:s0 + W])
            tags.append((i, s0))
    for tag, got, want in zip(tags, gots, G.oracle_many(jobs)):
        assert G.first_mismatch(got, want) == -1, "request %d window at %d" % tag


def test_config4_mix_per_request_keys_native_loop(P):
    """configs[3] at reduced count through the native closed loop: 1,500 requests, sizes log-uniform
    1-64 KiB with 0-15 B tails, per-request AES-128/256 keys expanded inside the loop, fully random
    ICBs, 256 in flight.  Every byte checked."""
    import gpu_util as G

    w = workloads.config4(n=1500)
    srcs = [G.to_device(w.payload(i)) for i in range(w.n)]
    dsts = [G.device_empty(int(w.length[i])) for i in range(w.n)]
    G.stream_sync()
    keys = np.zeros((w.n, 32), dtype=np.uint8)
    keybits = np.zeros(w.n, dtype=np.int32)
    for i in range(w.n):
        k = w.key_of(i)
        keys[i, : len(k)] = np.frombuffer(k, dtype=np.uint8)
        keybits[i] = 8 * len(k)
    r = P.aes_loop_run(w.icb, [s.data_ptr() for s in srcs], [d.data_ptr() for d in dsts], w.length,
                       window=w.in_flight, keys=keys, keybits=keybits)
    assert r["requests"] == w.n and r["bytes"] == w.total_bytes
    assert r["max_in_flight"] <= w.in_flight
    assert (r["lat_ns"] > 0).all()
    wants = G.oracle_many([(w.key_of(i), w.icb_of(i), w.payload(i)) for i in range(w.n)])
    for i in range(w.n):
        got = dsts[i].cpu().numpy()[: int(w.length[i])]
        assert G.first_mismatch(got, wants[i]) == -1, "request %d len %d" % (i, int(w.length[i]))


def test_buffer_reuse_sees_fresh_data(P):
    """The persistent kernel's L1 is never invalidated: a recycled src buffer must still be read
    fresh (payload loads are L2-only).  Same buffers, new contents, 20 rounds, in place and not."""
    import gpu_util as G

    torch = G.torch_cuda()
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7200]))
    key, n = rng.bytes(16), 48 * 1024 + 7
    ctx = P.aes_ctx_create(key)
    src, dst = G.device_empty(n), G.device_empty(n)
    from oracle import oracle as o

    for it in range(20):
        data = np.frombuffer(rng.bytes(n), dtype=np.uint8)
        icb = rng.bytes(16)
        src.copy_(torch.from_numpy(data))  # H2D memcpy, no kernel
        G.stream_sync()
        target = src if it % 2 else dst
        h = P.aes_ctr_submit(ctx, icb, src.data_ptr(), target.data_ptr(), n)
        P.aes_wait(h)
        assert G.first_mismatch(target.cpu().numpy(), o.ctr(key, icb, data)) == -1, "round %d" % it
    P.aes_ctx_destroy(ctx)


def test_host_resident_payload_zero_copy(P):
    """src/dst in pinned host memory (aes_host_alloc): the kernel reads and writes over PCIe; once
    aes_poll is true the host sees every byte."""
    from oracle import oracle as o

    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7300]))
    for keylen, n in ((16, 4096), (32, 100003), (16, 1 << 20)):
        key, icb = rng.bytes(keylen), rng.bytes(16)
        ps, pd = P.aes_host_alloc(n), P.aes_host_alloc(n)
        hs, hd = P.host_view(ps, n), P.host_view(pd, n)
        hs[:] = np.frombuffer(rng.bytes(n), dtype=np.uint8)
        hd[:] = 0
        ctx = P.aes_ctx_create(key)
        h = P.aes_ctr_submit(ctx, icb, ps, pd, n)
        P.aes_wait(h)
        want = o.ctr(key, icb, hs)
        assert hd.tobytes() == want
        P.aes_ctx_destroy(ctx)
        del hs, hd
        # freeing pinned memory synchronises the device: keep it until the engine stops (leak in test)


def test_ring_full_then_drains(P):
    """More submissions than ring slots: submit returns AES_E_AGAIN (never blocks), and every
    accepted request still completes with the right bytes."""
    from oracle import oracle as o
    import gpu_util as G

    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7400]))
    slots = P.aes_engine_info()["ring_slots"]
    key = rng.bytes(16)
    ctx = P.aes_ctx_create(key)
    n = 8 << 20
    big = G.to_device(np.frombuffer(rng.bytes(n), dtype=np.uint8))
    sink = G.device_empty(n)
    small_src = G.to_device(np.frombuffer(rng.bytes(256), dtype=np.uint8))
    small_dst = G.device_empty(256)
    G.stream_sync()
    handles, again = [], 0
    for i in range(slots + 64):
        try:
            handles.append(P.aes_ctr_submit(ctx, bytes(16), big.data_ptr(), sink.data_ptr(), n))
        except P.AesOffError as e:
            assert e.code == P.AES_E_AGAIN
            again += 1
    assert len(handles) + again == slots + 64
    icb = rng.bytes(16)
    while True:
        try:
            hs = P.aes_ctr_submit(ctx, icb, small_src.data_ptr(), small_dst.data_ptr(), 256)
            break
        except P.AesOffError as e:
            assert e.code == P.AES_E_AGAIN
    for h in handles + [hs]:
        P.aes_wait(h, 60_000_000_000)
    assert small_dst.cpu().numpy().tobytes() == o.ctr(key, icb, small_src.cpu().numpy())
    assert sink.cpu().numpy()[:4096].tobytes() == o.ctr(key, bytes(16), big[:4096].cpu().numpy())
    P.aes_ctx_destroy(ctx)


def test_many_threads_submit(P):
    """aes_ctr_submit from 8 executor threads at once (PAPER.md:350 '32-thread executor')."""
    import gpu_util as G

    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7500]))
    key = rng.bytes(32)
    ctx = P.aes_ctx_create(key)
    per, nthreads = 40, 8
    reqs = [(rng.bytes(16), np.frombuffer(rng.bytes(int(rng.integers(1, 20000))), dtype=np.uint8))
            for _ in range(per * nthreads)]
    srcs = [G.to_device(d) for _, d in reqs]
    dsts = [G.device_empty(len(d)) for _, d in reqs]
    G.stream_sync()
    errors = []

    def run(t):
        try:
            hs = []
            for i in range(t * per, (t + 1) * per):
                hs.append(P.aes_ctr_submit(ctx, reqs[i][0], srcs[i].data_ptr(), dsts[i].data_ptr(), len(reqs[i][1])))
            for h in hs:
                P.aes_wait(h)
        except Exception as e:  # noqa: BLE001
            errors.append(e)

    ts = [threading.Thread(target=run, args=(t,)) for t in range(nthreads)]
    [t.start() for t in ts]
    [t.join() for t in ts]
    assert not errors
    wants = G.oracle_many([(key, icb, d) for icb, d in reqs])
    for i, want in enumerate(wants):
        assert G.first_mismatch(dsts[i].cpu().numpy()[: len(reqs[i][1])], want) == -1, "request %d" % i
    P.aes_ctx_destroy(ctx)


def test_errors_and_handles(P):
    import gpu_util as G

    ctx = P.aes_ctx_create(bytes(16))
    buf = G.device_empty(4096)
    p = buf.data_ptr()
    for args, code in (((ctx, bytes(16), p + 4, p, 64), P.AES_E_ALIGN),
                       ((ctx, bytes(16), p, p + 32, 64), P.AES_E_OVERLAP),
                       ((0, bytes(16), p, p, 64), P.AES_E_INVAL)):
        with pytest.raises(P.AesOffError) as e:
            P.aes_ctr_submit(*args)
        assert e.value.code == code
    with pytest.raises(P.AesOffError) as e:
        P.aes_poll(1 << 60)  # never issued
    assert e.value.code == P.AES_E_INVAL
    with pytest.raises(P.AesOffError) as e:
        P.aes_ctr_launch_batch([ctx], bytes(16), [p], [p], [64])  # engine is running
    assert e.value.code == P.AES_E_BUSY
    h = P.aes_ctr_submit(ctx, bytes(16), 0, 0, 0)  # len 0: completes, touches nothing
    P.aes_wait(h)
    P.aes_ctx_destroy(ctx)


def test_context_key_paths(P):
    """How a key reaches the device (aesoff_internal.h): raw in the descriptor and expanded by the dispatcher
    warp (first and second submit of a context), by key-table index afterwards; indices rest after
    aes_ctx_destroy and run out -- the context then simply stays on the raw path."""
    import gpu_util as G
    from oracle import oracle as o

    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7600]))
    data = np.frombuffer(rng.bytes(4096 + 7), dtype=np.uint8)
    src = G.to_device(data)
    G.stream_sync()
    # (a) one context, six submits: raw, raw+install, four by index; both key sizes
    for keylen in (16, 24, 32):
        key = rng.bytes(keylen)
        ctx = P.aes_ctx_create(key)
        for j in range(6):
            icb = rng.bytes(16)
            dst = G.device_empty(len(data))
            P.aes_wait(P.aes_ctr_submit(ctx, icb, src.data_ptr(), dst.data_ptr(), len(data)))
            assert dst.cpu().numpy().tobytes() == o.ctr(key, icb, data), "submit %d of a %d-bit context" % (j, 8 * keylen)
        P.aes_ctx_destroy(ctx)
    # (b) 5,000 short-lived contexts (more than the key table has indices), three submits each, in flight together
    small = data[:80]
    ssrc = G.to_device(small)
    G.stream_sync()
    n_ctx, per = 5000, 3
    dsts = G.device_empty(n_ctx * per * 96)
    keys, icbs, hs = [], [], []
    for i in range(n_ctx):
        key = rng.bytes((16, 24, 32)[i % 3])
        ctx = P.aes_ctx_create(key)
        for j in range(per):
            icb = rng.bytes(16)
            while True:
                try:
                    hs.append(P.aes_ctr_submit(ctx, icb, ssrc.data_ptr(), dsts.data_ptr() + (i * per + j) * 96, len(small)))
                    break
                except P.AesOffError as e:
                    if e.code != P.AES_E_AGAIN:
                        raise
            keys.append(key)
            icbs.append(icb)
        P.aes_ctx_destroy(ctx)  # allowed as soon as the last submit has returned
    for h in hs:
        P.aes_wait(h)
    got = dsts.cpu().numpy()
    wants = G.oracle_many([(k, i, small) for k, i in zip(keys, icbs)])
    for r, want in enumerate(wants):
        assert got[r * 96: r * 96 + len(small)].tobytes() == want, "context %d submit %d" % (r // per, r % per)


def test_unit_sizes_half_rows_and_eighths(P):
    """The dispatcher's three unit sizes on one engine: a lone request is cut into 1/8-row units, a
    short queue of 1 MiB requests into half rows, a long queue into whole rows; every byte checked,
    ragged tails and an ICB whose low byte is not 0 (the first row starts in its middle)."""
    import time

    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7800]))
    key = rng.bytes(16)
    before = P.aes_engine_info()
    lone = [(key, rng.bytes(15) + b"\x9c", np.frombuffer(rng.bytes((1 << 20) + 7), dtype=np.uint8))]
    _check(P, lone)
    short = [(key, rng.bytes(15) + bytes([37 * i % 256]), np.frombuffer(rng.bytes((1 << 20) + 16 * i + 3), dtype=np.uint8))
             for i in range(6)]
    _check(P, short)
    long_q = [(key, rng.bytes(16), np.frombuffer(rng.bytes((2 << 20) + 5), dtype=np.uint8)) for i in range(48)]
    _check(P, long_q)
    time.sleep(0.01)  # the statistics are written when the dispatcher next finds the ring empty
    after = P.aes_engine_info()
    d = {k: after[k] - before[k] for k in ("cut_eighths", "cut_halves", "cut_rows")}
    assert sum(d.values()) == len(lone) + len(short) + len(long_q)
    if P.test_latency_units:
        # which size a request gets depends on the load it meets, i.e. on timing: the lone request finds the GPU
        # idle (1/8 rows); most of the 48 x 2 MiB queue must have been cut coarser than that
        assert d["cut_eighths"] >= 1 and d["cut_halves"] + d["cut_rows"] >= len(long_q) // 2, d
    else:
        assert d["cut_rows"] == sum(d.values())


def test_open_loop_executor_parity(P):
    """aes_openloop_run: 400 Poisson arrivals at 200 K requests/s, overlapping and blocking;
    every output byte against the oracle, latencies positive, nothing lost."""
    import gpu_util as G

    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7900]))
    n = 400
    key = rng.bytes(16)
    datas = [np.frombuffer(rng.bytes(int(rng.integers(1, 9000))), dtype=np.uint8) for _ in range(n)]
    icbs = rng.integers(0, 256, size=(n, 16), dtype=np.uint8)
    srcs = [G.to_device(d) for d in datas]
    arrival = np.cumsum(rng.exponential(1e9 / 200e3, size=n)).astype(np.uint64)
    wants = G.oracle_many([(key, icbs[i].tobytes(), datas[i]) for i in range(n)])
    ctx = P.aes_ctx_create(key)
    for blocking in (False, True):
        dsts = [G.device_empty(len(d)) for d in datas]
        G.stream_sync()
        r = P.aes_openloop_run(icbs, [s.data_ptr() for s in srcs], [d.data_ptr() for d in dsts], [len(d) for d in datas],
                               arrival, ctx, blocking=blocking)
        assert r["requests"] == n and r["bytes"] == sum(len(d) for d in datas)
        assert (r["lat_ns"] > 0).all()
        assert r["elapsed_ns"] >= int(arrival[-1])  # nothing is submitted before it arrives
        for i in range(n):
            assert G.first_mismatch(dsts[i].cpu().numpy()[: len(datas[i])], wants[i]) == -1, "request %d" % i
    P.aes_ctx_destroy(ctx)


def test_closed_loop_from_four_threads(P):
    """aes_loop_run_mt: four executor threads share the ring ("worker pool"); every byte checked."""
    import gpu_util as G

    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 8000]))
    n = 600
    key = rng.bytes(32)
    datas = [np.frombuffer(rng.bytes(int(rng.integers(1, 30000))), dtype=np.uint8) for _ in range(n)]
    icbs = rng.integers(0, 256, size=(n, 16), dtype=np.uint8)
    srcs = [G.to_device(d) for d in datas]
    dsts = [G.device_empty(len(d)) for d in datas]
    G.stream_sync()
    ctx = P.aes_ctx_create(key)
    r = P.aes_loop_run(icbs, [s.data_ptr() for s in srcs], [d.data_ptr() for d in dsts], [len(d) for d in datas],
                       window=64, ctx=ctx, threads=4)
    assert r["requests"] == n and r["bytes"] == sum(len(d) for d in datas) and (r["lat_ns"] > 0).all()
    wants = G.oracle_many([(key, icbs[i].tobytes(), datas[i]) for i in range(n)])
    for i in range(n):
        assert G.first_mismatch(dsts[i].cpu().numpy()[: len(datas[i])], wants[i]) == -1, "request %d" % i
    P.aes_ctx_destroy(ctx)

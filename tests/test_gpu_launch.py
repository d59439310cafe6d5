"""-m gpu parity, launch backend (aes_ctr_launch_batch): the CUDA path against the oracle,
byte for byte (bit-exact: AES-CTR has one correct output).

The launch backend runs exactly the worker code of the persistent engine from an ordinary kernel
launch, so these cases pin the arithmetic (counter blocks, rounds, tails, chunking) independently of
the ring/mailbox machinery, which tests/test_gpu_engine.py covers.
"""
import numpy as np
import pytest

from paper_2607_02630_b200 import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import paper_2607_02630_b200.binding as B

    return B


def _run_batch(P, reqs, chunk_rows=0, in_place=False):
    """reqs: list of (key, icb, payload ndarray).  Returns list of output ndarrays."""
    import gpu_util as G

    ctxs = {}
    srcs, dsts, handles = [], [], []
    for key, icb, data in reqs:
        if key not in ctxs:
            ctxs[key] = P.aes_ctx_create(key)
        s = G.to_device(data) if len(data) else G.device_empty(0)
        d = s if in_place else G.device_empty(len(data))
        srcs.append(s)
        dsts.append(d)
    G.stream_sync()
    P.aes_ctr_launch_batch([ctxs[k] for k, _, _ in reqs], b"".join(icb for _, icb, _ in reqs),
                           [s.data_ptr() for s in srcs], [d.data_ptr() for d in dsts],
                           [len(x) for _, _, x in reqs], cuda_stream=0, chunk_rows=chunk_rows)
    G.torch_cuda().cuda.synchronize()  # no persistent engine in this module: a device sync is fine
    outs = [d.cpu().numpy()[: len(x)] for d, (_, _, x) in zip(dsts, reqs)]
    for c in ctxs.values():
        P.aes_ctx_destroy(c)
    return outs


def _check(P, reqs, **kw):
    import gpu_util as G

    outs = _run_batch(P, reqs, **kw)
    wants = G.oracle_many([(k, i, d) for k, i, d in reqs])
    for n, (got, want) in enumerate(zip(outs, wants)):
        bad = G.first_mismatch(got, want)
        assert bad == -1, "request %d (len %d, keybits %d, icb %s): first mismatch at byte %d" % (
            n, len(reqs[n][2]), 8 * len(reqs[n][0]), reqs[n][1].hex(), bad)


def test_config1_aes128_64KiB(P):
    w = workloads.config1()
    _check(P, [(w.key_of(0), w.icb_of(0), w.payload(0))])


@pytest.mark.parametrize("keylen", [16, 24, 32])
def test_lengths_tails_and_tiles(P, keylen):
    """Empty, sub-block, block +-1, row (4 KiB) +-1, chunk (16 KiB) +-1, several chunks + ragged tail."""
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 1000 + keylen]))
    key = rng.bytes(keylen)
    lens = [0, 1, 15, 16, 17, 31, 32, 33, 255, 256, 4095, 4096, 4097, 4111, 16383, 16384, 16385,
            65536 + 5, 3 * 16384 + 16 * 77 + 9, (1 << 20) + 5]
    reqs = []
    for n in lens:
        icb = rng.bytes(8) + bytes(8)
        reqs.append((key, icb, np.frombuffer(rng.bytes(n), dtype=np.uint8)))
    _check(P, reqs)


@pytest.mark.parametrize("keylen", [16, 24, 32])
def test_counter_carries(P, keylen):
    """R4: the counter is a 128-bit big-endian integer; carries out of the low 8/32/64/128 bits, both
    on the first increment and in the middle of a chunk, and ICBs whose last byte is not zero (rows
    are aligned on that byte)."""
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 2000 + keylen]))
    key = rng.bytes(keylen)
    reqs = []
    for icb in workloads.edge_icbs():
        for n in (16 * 600 + 3, 16 * 70, 40000):
            reqs.append((key, icb, np.frombuffer(rng.bytes(n), dtype=np.uint8)))
    for last in (1, 31, 32, 33, 128, 254, 255):
        icb = rng.bytes(15) + bytes([last])
        for n in (5, 16 * (256 - last), 16 * (256 - last) + 1, 16 * 300 + 7, 70001):
            reqs.append((key, icb, np.frombuffer(rng.bytes(n), dtype=np.uint8)))
    _check(P, reqs)


@pytest.mark.parametrize("chunk_rows", [1, 2, 16, 64])
def test_chunk_sizes(P, chunk_rows):
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 3000 + chunk_rows]))
    reqs = []
    for keylen, n in ((16, 300000 + 7), (32, 1 << 19), (16, 4096 * 64 + 16), (32, 100)):
        reqs.append((rng.bytes(keylen), rng.bytes(16), np.frombuffer(rng.bytes(n), dtype=np.uint8)))
    _check(P, reqs, chunk_rows=chunk_rows)


def test_in_place_and_mixed_keys(P):
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 4000]))
    reqs = [(rng.bytes(16 if i % 2 else 32), rng.bytes(16), np.frombuffer(rng.bytes(1000 * i + i), dtype=np.uint8))
            for i in range(1, 40)]
    _check(P, reqs, in_place=True)


def test_decrypt_is_encrypt(P):
    """CTR is an involution (SP 800-38A 6.5): running the output through again returns the input."""
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 5000]))
    key, icb = rng.bytes(32), rng.bytes(16)
    data = np.frombuffer(rng.bytes(123457), dtype=np.uint8)
    (ct,) = _run_batch(P, [(key, icb, data)])
    (pt,) = _run_batch(P, [(key, icb, ct)])
    assert np.array_equal(pt, data) and not np.array_equal(ct, data)


def test_large_request_sampled_windows(P):
    """64 MiB AES-256 (the sweep's largest size): too long for the byte-level oracle in full, so check
    sampled 64 KiB windows with oracle_ctr_at, always including the first and the last block."""
    import gpu_util as G

    torch = G.torch_cuda()
    n = 64 << 20
    g = torch.Generator(device="cuda:0").manual_seed(workloads.SEED_BASE + 5)
    src = torch.randint(0, 256, (n,), dtype=torch.uint8, device="cuda:0", generator=g)
    dst = torch.empty_like(src)
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 6000]))
    key, icb = rng.bytes(32), rng.bytes(16)
    ctx = P.aes_ctx_create(key)
    torch.cuda.synchronize()
    P.aes_ctr_launch_batch([ctx], icb, [src.data_ptr()], [dst.data_ptr()], [n])
    torch.cuda.synchronize()
    P.aes_ctx_destroy(ctx)
    W = 64 << 10
    starts = [0, n - W] + [int(x) * 16 for x in rng.integers(0, (n - W) // 16, size=10)]
    jobs, gots = [], []
    for s0 in starts:
        jobs.append((key, icb, src[s0:s0 + W].cpu().numpy(), s0 // 16))
        gots.append(dst[s0:s0 + W].cpu().numpy())
    for s0, got, want in zip(starts, gots, G.oracle_many(jobs)):
        assert G.first_mismatch(got, want) == -1, "window at %d" % s0


def test_errors_launch(P):
    import gpu_util as G

    ctx = P.aes_ctx_create(bytes(16))
    buf = G.device_empty(4096)
    p = buf.data_ptr()
    with pytest.raises(P.AesOffError) as e:
        P.aes_ctr_launch_batch([ctx], bytes(16), [p + 1], [p + 1], [64])
    assert e.value.code == P.AES_E_ALIGN
    with pytest.raises(P.AesOffError) as e:
        P.aes_ctr_launch_batch([ctx], bytes(16), [p], [p + 16], [64])
    assert e.value.code == P.AES_E_OVERLAP
    with pytest.raises(P.AesOffError) as e:
        P.aes_ctr_launch_batch([0], bytes(16), [p], [p], [64])
    assert e.value.code == P.AES_E_INVAL
    P.aes_ctx_destroy(ctx)


def test_calibration_microkernels(P):
    """aes_calibrate: the lookup pipe delivers (nearly) its nominal 32 lookups per clock per SM with the engine's
    table layout -- i.e. the layout is conflict-free in fact, not only by construction -- and the ALU pipe its
    nominal 2 warp-wide instructions; the numbers bench.py's roofline stands on."""
    c = P.aes_calibrate(0)
    assert c["sm_count"] >= 100
    assert 28.0 <= c["lookups_per_clk_per_sm"] <= 32.5, c
    assert 26.0 <= c["round_lookups_per_clk_per_sm"] <= 32.5, c
    assert 1.7 <= c["alu_instr_per_clk_per_sm"] <= 2.1, c
    assert c["copy_gbs"] > 3000.0, c
    # the bitsliced S-box the table form was chosen against: the generated circuit is right on all 256 inputs, and at
    # 117 LOP3 per evaluation it cannot run faster than the ALU pipe allows (2 warp-wide instructions per clock per SM)
    assert c["bitslice_mismatches"] == 0, c
    assert 0.005 <= c["bitslice_sboxes_per_clk_per_sm"] <= 2.1 / 117.0 * 1.05, c


@pytest.mark.parametrize("low4", ["01fffe00", "01ffff00", "ffffff37", "ffffffff", "00000000", "a1b2ff9c"])
def test_consecutive_rows_and_carries_out_of_counter_byte_14(P, low4):
    """Whole-row units are two consecutive rows; the second row's set-up is derived from the first's unless the
    increment carries out of counter byte 14.  96 MiB in one launch (the first 12,000 rows run as whole-row units),
    ICBs whose bytes 12..15 put that carry on the first, the second, or no row of a unit, and a ragged first row:
    the first 2 MiB in full and sampled windows against the oracle."""
    import gpu_util as G

    torch = G.torch_cuda()
    n = (96 << 20) + 11
    g = torch.Generator(device="cuda:0").manual_seed(workloads.SEED_BASE + 77)
    src = torch.randint(0, 256, (n,), dtype=torch.uint8, device="cuda:0", generator=g)
    dst = torch.empty_like(src)
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 6100]))
    key = rng.bytes(16)
    icb = rng.bytes(12) + bytes.fromhex(low4)
    if low4 == "ffffffff":
        icb = b"\xff" * 16  # the whole 128-bit counter wraps on the first increment
    ctx = P.aes_ctx_create(key)
    torch.cuda.synchronize()
    P.aes_ctr_launch_batch([ctx], icb, [src.data_ptr()], [dst.data_ptr()], [n])
    torch.cuda.synchronize()
    P.aes_ctx_destroy(ctx)
    W = 64 << 10
    starts = list(range(0, 2 << 20, W)) + [n - W - 11] + [int(x) * 16 for x in rng.integers(0, (40 << 20) // 16, size=12)]
    jobs, gots = [], []
    for s0 in starts:
        e0 = min(n, s0 + W + (11 if s0 == n - W - 11 else 0))
        jobs.append((key, icb, src[s0:e0].cpu().numpy(), s0 // 16))
        gots.append(dst[s0:e0].cpu().numpy())
    for s0, got, want in zip(starts, gots, G.oracle_many(jobs)):
        assert G.first_mismatch(got, want) == -1, "window at %d" % s0


def test_launches_on_two_streams_do_not_trample_each_other(P):
    """aes_ctr_launch_batch keeps ONE device blob of descriptors, keys and tickets; calls on different streams are
    serialised on the device through an event (the second call's copy waits for the first call's kernel).  Two streams
    alternating, several calls each, nothing synchronised in between; every byte against the oracle."""
    import gpu_util as G

    torch = G.torch_cuda()
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 6900]))
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    keys = [rng.bytes(16), rng.bytes(32)]
    ctxs = [P.aes_ctx_create(k) for k in keys]
    calls = []
    for c in range(8):
        n = 3 + c % 3
        datas = [np.frombuffer(rng.bytes(int(rng.integers(1, 300000))), dtype=np.uint8) for _ in range(n)]
        icbs = [rng.bytes(16) for _ in range(n)]
        srcs = [G.to_device(d) for d in datas]
        dsts = [G.device_empty(len(d)) for d in datas]
        calls.append((c % 2, datas, icbs, srcs, dsts))
    torch.cuda.synchronize()
    for which, datas, icbs, srcs, dsts in calls:
        P.aes_ctr_launch_batch([ctxs[which]] * len(datas), b"".join(icbs), [s.data_ptr() for s in srcs],
                               [d.data_ptr() for d in dsts], [len(d) for d in datas], cuda_stream=streams[which].cuda_stream)
    for s in streams:
        s.synchronize()
    jobs, gots = [], []
    for which, datas, icbs, srcs, dsts in calls:
        for d, i, out in zip(datas, icbs, dsts):
            jobs.append((keys[which], i, d))
            gots.append(out.cpu().numpy()[:len(d)])
    for k, (got, want) in enumerate(zip(gots, G.oracle_many(jobs))):
        assert G.first_mismatch(got, want) == -1, "request %d" % k
    for c in ctxs:
        P.aes_ctx_destroy(c)

"""-m gpu: ECB and CBC-decrypt on the engine and through ordinary launches (SP 800-38A
sec. 6.1, 6.2), byte for byte against the oracle's ECB / CBC (pinned in tests/test_oracle_modes.py to the F.1 / F.2
printed vectors and to two libraries).  Decryption runs the equivalent inverse cipher (FIPS-197 sec. 5.3.5) out of the
Td0 table; CTR requests share batches with the other modes."""
import numpy as np
import pytest

from paper_2607_02630_b200 import workloads

pytestmark = pytest.mark.gpu

LENS = [0, 16, 32, 4080, 4096, 4112, 16384 + 16, 65536, 65536 + 4096 + 16, (1 << 20) + 48, 3 * (1 << 20)]


def _want(o, mode, key, iv, data):
    if mode == 0:
        return o.ctr(key, iv, data)
    if mode == 1:
        return o.ecb_encrypt(key, data)
    if mode == 2:
        return o.ecb_decrypt(key, data)
    return o.cbc_decrypt(key, iv, data)


def _cases(rng, keylens=(16, 24, 32)):
    cases = []
    for kl in keylens:
        key = rng.bytes(kl)
        for mode in (1, 2, 3):
            for n in (LENS if kl == 16 else LENS[:-2]):   # the two longest once per mode
                cases.append((mode, key, rng.bytes(16), np.frombuffer(rng.bytes(n), dtype=np.uint8)))
        cases.append((0, key, rng.bytes(16), np.frombuffer(rng.bytes(70001), dtype=np.uint8)))  # CTR in the same batch
    return cases


def _check(outs, cases):
    import concurrent.futures as cf
    import os

    import gpu_util as G
    from oracle import oracle as o

    with cf.ThreadPoolExecutor(max(1, len(os.sched_getaffinity(0)))) as ex:   # the C oracle releases the GIL
        wants = list(ex.map(lambda c: _want(o, c[0], c[1], c[2], c[3]), cases))
    for i, ((mode, key, iv, data), got, want) in enumerate(zip(cases, outs, wants)):
        bad = G.first_mismatch(got, want)
        assert bad == -1, "case %d: mode %d, %d-bit key, len %d: first mismatch at byte %d" % (i, mode, 8 * len(key), len(data), bad)


@pytest.mark.parametrize("chunk_rows", [0, 1, 16])
def test_modes_through_ordinary_launches(chunk_rows):
    import gpu_util as G
    import paper_2607_02630_b200.binding as B

    torch = G.torch_cuda()
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 8300 + chunk_rows]))
    cases = _cases(rng)
    ctxs = {}
    srcs = [G.to_device(d) if len(d) else G.device_empty(0) for _, _, _, d in cases]
    dsts = [G.device_empty(len(d)) for _, _, _, d in cases]
    for _, key, _, _ in cases:
        ctxs.setdefault(key, B.aes_ctx_create(key))
    torch.cuda.synchronize()
    B.aes_mode_launch_batch([m for m, _, _, _ in cases], [ctxs[k] for _, k, _, _ in cases], b"".join(iv for _, _, iv, _ in cases),
                            [s.data_ptr() for s in srcs], [d.data_ptr() for d in dsts], [len(d) for _, _, _, d in cases],
                            chunk_rows=chunk_rows)
    torch.cuda.synchronize()
    _check([d.cpu().numpy()[:len(c[3])] for d, c in zip(dsts, cases)], cases)
    for c in ctxs.values():
        B.aes_ctx_destroy(c)


@pytest.fixture(scope="module", params=["latency_units", "row_units_only"])
def E(request):
    import gpu_util as G
    import paper_2607_02630_b200.binding as B

    torch = G.torch_cuda()
    torch.zeros(1, device="cuda:0")
    torch.cuda.synchronize()
    B.aes_engine_start(0, idle_exit_ms=60000, fine_rows=0 if request.param == "latency_units" else B.AES_FINE_ROWS_OFF)
    yield B
    B.aes_engine_stop()


def _submit(E, ctx, mode, iv, s, d, n):
    if mode == 0:
        return E.aes_ctr_submit(ctx, iv, s, d, n)
    if mode == 3:
        return E.aes_cbc_decrypt_submit(ctx, iv, s, d, n)
    return E.aes_ecb_submit(ctx, mode == 2, s, d, n)


def test_modes_on_the_engine(E):
    import gpu_util as G

    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 8400]))
    cases = _cases(rng)
    ctxs = {}
    srcs = [G.to_device(d) if len(d) else G.device_empty(0) for _, _, _, d in cases]
    dsts = [G.device_empty(len(d)) for _, _, _, d in cases]
    G.stream_sync()
    hs = []
    for (mode, key, iv, data), s, d in zip(cases, srcs, dsts):
        if key not in ctxs:
            ctxs[key] = E.aes_ctx_create(key)
        hs.append(_submit(E, ctxs[key], mode, iv, s.data_ptr(), d.data_ptr(), len(data)))
    for h in hs:
        E.aes_wait(h, 20_000_000_000)
    _check([d.cpu().numpy()[:len(c[3])] for d, c in zip(dsts, cases)], cases)
    # a long queue of decrypting requests (whole-row units), then lone ones (1/8-row units)
    key, iv = rng.bytes(32), rng.bytes(16)
    big = [(3 if i % 2 else 2, key, iv, np.frombuffer(rng.bytes(2 << 20), dtype=np.uint8)) for i in range(40)]
    bs = [G.to_device(c[3]) for c in big]
    bd = [G.device_empty(len(c[3])) for c in big]
    G.stream_sync()
    ctx = E.aes_ctx_create(key)
    hs = [_submit(E, ctx, c[0], c[2], s.data_ptr(), d.data_ptr(), len(c[3])) for c, s, d in zip(big, bs, bd)]
    for h in hs:
        E.aes_wait(h, 20_000_000_000)
    _check([d.cpu().numpy() for d in bd], big)
    for c, s, d in list(zip(big, bs, bd))[:3]:
        E.aes_wait(_submit(E, ctx, c[0], c[2], s.data_ptr(), d.data_ptr(), len(c[3])), 20_000_000_000)
        _check([d.cpu().numpy()], [c])
    # ECB may run in place; a round trip gives the plaintext back
    p = np.frombuffer(rng.bytes(100000 - 100000 % 16), dtype=np.uint8)
    t = G.to_device(p)
    G.stream_sync()
    E.aes_wait(E.aes_ecb_submit(ctx, False, t.data_ptr(), t.data_ptr(), len(p)))
    E.aes_wait(E.aes_ecb_submit(ctx, True, t.data_ptr(), t.data_ptr(), len(p)))
    assert G.first_mismatch(t.cpu().numpy(), p.tobytes()) == -1
    E.aes_ctx_destroy(ctx)
    for c in ctxs.values():
        E.aes_ctx_destroy(c)


def test_mode_errors(E):
    import gpu_util as G

    t = G.device_empty(4096)
    ctx = E.aes_ctx_create(bytes(16))
    with pytest.raises(E.AesOffError) as e:
        E.aes_ecb_submit(ctx, False, t.data_ptr(), t.data_ptr() + 2048, 100)      # not whole blocks
    assert e.value.code == E.AES_E_INVAL
    with pytest.raises(E.AesOffError) as e:
        E.aes_cbc_decrypt_submit(ctx, bytes(16), t.data_ptr(), t.data_ptr(), 1024)  # in place
    assert e.value.code == E.AES_E_OVERLAP
    with pytest.raises(E.AesOffError) as e:
        E.aes_cbc_decrypt_submit(ctx, bytes(16), t.data_ptr(), t.data_ptr() + 16, 1024)
    assert e.value.code == E.AES_E_OVERLAP
    E.aes_ctx_destroy(ctx)


"""aes_ctr_launch_static: the launch backend for callers that must not allocate (include/aesoff.h).

Who needs it: a server whose own pool already holds all of the GPU's memory (cudaMalloc fails there), a process
with a never-ending kernel on the GPU -- this library's persistent engine is one -- where cudaFree would wait for
ever, and request handlers that cannot pay a cudaMalloc in front of a 4 KiB offload.  The entry point keeps its
whole queue in a 19.25 KiB static device array of the library instead, and so takes at most AES_STATIC_MAX_BYTES.

What is checked: on the same inputs, its output equals, byte for byte, the output of the existing path
(aes_ctr_launch_batch, which cudaMallocs its queue) and, for the sizes the oracle finishes quickly, the oracle's;
calls follow each other on one stream WITHOUT a synchronisation in between, a large request first and small ones
after it, so that whatever the earlier call left in the shared array (more tickets, another key, another
descriptor) would show up in the later ones if the set-up kernel did not rewrite it.

This file sorts last on purpose (`pytest --collect-only`): with `-x` a failure here hides no other test.
It needs nothing from the other tests and leaves nothing behind: it runs alone in a fresh process, where its first
call also performs the per-device set-up, and after the rest of the suite alike.
"""
import numpy as np
import pytest

from paper_2607_02630_b200 import workloads


@pytest.fixture(scope="module")
def P():
    import paper_2607_02630_b200.binding as B

    return B


def _cases():
    """(key, icb, length): big before small; ragged tails; ICBs whose low counter byte is not zero (rows then
    start inside the payload) and one that carries out of the low 32 bits; all three key sizes."""
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7700]))
    k256, k128, k192 = rng.bytes(32), rng.bytes(16), rng.bytes(24)
    return [
        (k256, rng.bytes(15) + b"\x9d", (1 << 20) + 5),                      # 257 rows, 65 tickets
        (k128, rng.bytes(12) + b"\xff\xff\xff\xf0", 4096 + 17),              # 2 rows, 1 ticket, 32-bit carry inside
        (k192, rng.bytes(8) + bytes(8), 16),                                  # one block
        (k128, rng.bytes(8) + bytes(7) + b"\x01", 3 * 16384 + 16 * 77 + 9),   # several chunks + ragged tail
    ]


@pytest.mark.gpu
def test_static_scratch_path_equals_existing_path_on_calls_in_a_row(P):
    import gpu_util as G

    torch = G.torch_cuda()
    if P.aes_engine_info()["running"]:  # an earlier module's engine would make both launch backends AES_E_BUSY
        P.aes_engine_stop()
    cases = _cases()
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7701]))
    data = [np.frombuffer(rng.bytes(n), dtype=np.uint8) for _, _, n in cases]
    ctxs = [P.aes_ctx_create(k) for k, _, _ in cases]
    srcs = [G.to_device(x) for x in data]
    got = [G.device_empty(len(x) + 64) for x in data]   # 64 marker bytes behind each output
    ref = [G.device_empty(len(x)) for x in data]
    for g in got:
        g.fill_(0xA5)
    torch.cuda.synchronize()

    # the new entry point: every call in a row on the legacy default stream, nothing in between
    for c, (_, icb, n), s, g in zip(ctxs, cases, srcs, got):
        P.aes_ctr_launch_static(c, icb, s.data_ptr(), g.data_ptr(), n, device=0, cuda_stream=0)
    torch.cuda.synchronize()
    # the existing path on the same inputs
    P.aes_ctr_launch_batch(ctxs, b"".join(icb for _, icb, _ in cases), [s.data_ptr() for s in srcs],
                           [r.data_ptr() for r in ref], [n for _, _, n in cases], cuda_stream=0)
    torch.cuda.synchronize()

    wants = G.oracle_many([(k, icb, x) for (k, icb, _), x in zip(cases, data)])
    for i, ((_, icb, n), g, r, want) in enumerate(zip(cases, got, ref, wants)):
        out = g.cpu().numpy()
        assert np.array_equal(out[:n], r.cpu().numpy()[:n]), "call %d (len %d): differs from aes_ctr_launch_batch" % (i, n)
        assert G.first_mismatch(out[:n], want) == -1, "call %d (len %d, icb %s): differs from the oracle" % (i, n, icb.hex())
        assert (out[n:] == 0xA5).all(), "call %d wrote past the end of dst" % i

    # once more, in place, on a stream of the caller's own, the calls in the opposite order (small before big)
    st = torch.cuda.Stream()
    inpl = [G.to_device(x) for x in data]
    torch.cuda.synchronize()
    for c, (_, icb, n), b in reversed(list(zip(ctxs, cases, inpl))):
        P.aes_ctr_launch_static(c, icb, b.data_ptr(), b.data_ptr(), n, device=0, cuda_stream=st.cuda_stream)
    st.synchronize()
    for i, (b, r) in enumerate(zip(inpl, ref)):
        assert torch.equal(b, r[: b.numel()]), "in-place call %d differs from aes_ctr_launch_batch" % i
    for c in ctxs:
        P.aes_ctx_destroy(c)


@pytest.mark.gpu
def test_static_scratch_path_at_its_maximum_size(P):
    """AES_STATIC_MAX_BYTES with a non-zero low counter byte is the request that needs the most tickets the array
    offers (16,385 rows in chunks of 32); a 4 KiB call follows it at once.  Against the existing path."""
    import gpu_util as G

    torch = G.torch_cuda()
    if P.aes_engine_info()["running"]:
        P.aes_engine_stop()
    n = P.AES_STATIC_MAX_BYTES
    gen = torch.Generator(device="cuda:0").manual_seed(workloads.SEED_BASE + 7702)
    src = torch.randint(0, 256, (n,), dtype=torch.uint8, device="cuda:0", generator=gen)
    got, ref = G.device_empty(n), G.device_empty(n)
    got_small, ref_small = G.device_empty(4096), G.device_empty(4096)
    key, icb = bytes(range(16)), bytes(range(100, 115)) + b"\xfe"
    ctx = P.aes_ctx_create(key)
    torch.cuda.synchronize()
    P.aes_ctr_launch_static(ctx, icb, src.data_ptr(), got.data_ptr(), n)
    P.aes_ctr_launch_static(ctx, icb, src.data_ptr(), got_small.data_ptr(), 4096)
    torch.cuda.synchronize()
    P.aes_ctr_launch_batch([ctx, ctx], icb + icb, [src.data_ptr()] * 2, [ref.data_ptr(), ref_small.data_ptr()], [n, 4096])
    torch.cuda.synchronize()
    assert torch.equal(got, ref)
    assert torch.equal(got_small, ref_small)
    assert not torch.equal(got[:4096], src[:4096])  # something was computed
    P.aes_ctx_destroy(ctx)


def test_static_scratch_path_refuses_what_does_not_fit(P):
    """Beyond AES_STATIC_MAX_BYTES the call fails with AES_E_TOOBIG before it touches CUDA (so this runs without a GPU):
    the array cannot grow, and growing is exactly what this entry point's callers cannot do."""
    ctx = P.aes_ctx_create(bytes(16))
    with pytest.raises(P.AesOffError) as e:
        P.aes_ctr_launch_static(ctx, bytes(16), 4096, 4096, P.AES_STATIC_MAX_BYTES + 1)
    assert e.value.code == P.AES_E_TOOBIG and "AES_STATIC_MAX_BYTES" in str(e.value)
    assert P.aes_last_error() == P.AES_E_TOOBIG
    with pytest.raises(P.AesOffError) as e:
        P.aes_ctr_launch_static(ctx, bytes(16), 4096 + 8, 4096, 64)
    assert e.value.code == P.AES_E_ALIGN
    with pytest.raises(P.AesOffError) as e:
        P.aes_ctr_launch_static(ctx, bytes(16), 4096, 4096 + 16, 64)
    assert e.value.code == P.AES_E_OVERLAP
    P.aes_ctr_launch_static(ctx, bytes(16), 0, 0, 0)  # an empty request completes without touching anything
    P.aes_ctx_destroy(ctx)

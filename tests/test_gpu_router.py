"""-m gpu: the request router against REAL addresses (csrc/aesoff_runtime.cpp route()).

tests/test_router_cpu.py covers the decision table and the page cache over a synthetic address map.  Here the owner of a
buffer comes from cudaPointerGetAttributes:
  - on ONE GPU, with the test hook AESOFF_ROUTE_ALWAYS=1 (read at aes_engine_start) that switches off the "one engine on a
    one-GPU node: look at nothing" shortcut, so that device, pinned-host and registered-host addresses all pass through
    resolve_owner + the per-thread page cache;
  - on TWO GPUs (skipped below two): one engine each in one process, one shared context, requests whose buffers live on
    GPU 0, on GPU 1 and in pinned host memory, handles of both engines polled from one loop, a request whose src and dst
    belong to different GPUs refused with AES_E_INVAL, aes_engine_stop_device(1) while engine 0 keeps serving.
Every output byte is compared with the oracle ("each offload belongs to one request": no exchange).
"""
import os

import numpy as np
import pytest

from paper_2607_02630_b200 import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture()
def P():
    import paper_2607_02630_b200.binding as B

    if B.aes_engine_info()["engines_running"]:
        B.aes_engine_stop()
    yield B
    os.environ.pop("AESOFF_ROUTE_ALWAYS", None)
    if B.aes_engine_info()["engines_running"]:
        B.aes_engine_stop()


def _wait_all(P, hs):
    pending = list(hs)
    for _ in range(2_000_000):  # one loop over handles of whatever engine
        pending = [h for h in pending if not P.aes_poll(h)]
        if not pending:
            return
    raise AssertionError("%d requests did not complete" % len(pending))


def test_forced_lookup_on_one_gpu(P):
    import gpu_util as G
    from oracle import oracle as o

    torch = G.torch_cuda()
    torch.zeros(1, device="cuda:0")
    torch.cuda.synchronize()
    os.environ["AESOFF_ROUTE_ALWAYS"] = "1"
    P.aes_engine_start(0, idle_exit_ms=60000)
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 8800]))
    key = rng.bytes(32)
    ctx = P.aes_ctx_create(key)
    n = 70_000 + 9
    data = [np.frombuffer(rng.bytes(n), dtype=np.uint8) for _ in range(6)]
    icbs = [rng.bytes(16) for _ in range(6)]
    dev_src = [G.to_device(x) for x in data]
    dev_dst = [G.device_empty(n) for _ in data]
    hp = [P.aes_host_alloc(n) for _ in range(4)]             # pinned, GPU-addressable host memory
    own = np.zeros(n + 64, dtype=np.uint8)                    # the server's own buffer, registered in place
    own_addr = (own.ctypes.data + 15) & ~15
    P.aes_host_register(own_addr, n)
    own_view = own[own_addr - own.ctypes.data: own_addr - own.ctypes.data + n]
    G.stream_sync()
    for i in (2, 3):
        P.host_view(hp[i - 2], n)[:] = data[i]
    own_view[:] = data[5]
    try:
        for sweep in range(2):  # second sweep: every page is remembered; then once more after a flush
            hs = [
                P.aes_ctr_submit(ctx, icbs[0], dev_src[0].data_ptr(), dev_dst[0].data_ptr(), n),   # device -> device
                P.aes_ctr_submit(ctx, icbs[1], dev_src[1].data_ptr(), dev_src[1].data_ptr(), n) if sweep == 0 else
                P.aes_ctr_submit(ctx, icbs[1], dev_src[1].data_ptr(), dev_src[1].data_ptr(), 0),   # in place (once)
                P.aes_ctr_submit(ctx, icbs[2], hp[0], hp[2], n),                                   # host -> host
                P.aes_ctr_submit(ctx, icbs[3], hp[1], dev_dst[3].data_ptr(), n),                   # host -> device
                P.aes_ctr_submit(ctx, icbs[4], dev_src[4].data_ptr(), hp[3], n),                   # device -> host
                P.aes_ctr_submit(ctx, icbs[5], own_addr, dev_dst[5].data_ptr(), n),                # registered -> device
            ]
            assert all(h >> 56 == 0 for h in hs)
            _wait_all(P, hs)
            outs = {0: dev_dst[0].cpu().numpy(), 1: dev_src[1].cpu().numpy(), 2: P.host_view(hp[2], n).copy(),
                    3: dev_dst[3].cpu().numpy(), 4: P.host_view(hp[3], n).copy(), 5: dev_dst[5].cpu().numpy()}
            for i, got in outs.items():
                assert G.first_mismatch(got, o.ctr(key, icbs[i], data[i])) == -1, "sweep %d request %d" % (sweep, i)
            P.aes_route_flush()
        assert P.aes_engine_info()["running"] == 1
    finally:
        P.aes_engine_stop()
        P.aes_host_unregister(own_addr)
        for p in hp:
            P.aes_host_free(p)
        P.aes_ctx_destroy(ctx)


def test_two_engines_in_one_process(P):
    import gpu_util as G
    from oracle import oracle as o

    torch = G.torch_cuda()
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs: one engine each")
    for d in (0, 1):
        torch.zeros(1, device="cuda:%d" % d)
        torch.cuda.synchronize(d)
    torch.cuda.set_device(0)
    P.aes_engine_start(0, idle_exit_ms=60000)
    P.aes_engine_start(1, idle_exit_ms=60000)
    assert torch.cuda.current_device() == 0, "aes_engine_start must leave the caller's device alone"
    assert P.aes_engine_info()["engines_running"] == 2
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 8801]))
    key = rng.bytes(16)
    ctx = P.aes_ctx_create(key)  # one context, both engines (its key is filed per engine)
    n = (1 << 20) + 5
    data = [np.frombuffer(rng.bytes(n), dtype=np.uint8) for _ in range(4)]
    icbs = [rng.bytes(16) for _ in range(4)]
    src0 = torch.from_numpy(np.array(data[0])).to("cuda:0")
    dst0 = torch.empty(n, dtype=torch.uint8, device="cuda:0")
    src1 = torch.from_numpy(np.array(data[1])).to("cuda:1")
    dst1 = torch.empty(n, dtype=torch.uint8, device="cuda:1")
    hsrc, hdst_a, hdst_b = P.aes_host_alloc(n), P.aes_host_alloc(n), P.aes_host_alloc(n)
    P.host_view(hsrc, n)[:] = data[2]
    for d in (0, 1):
        torch.cuda.current_stream(d).synchronize()
    try:
        for rep in range(3):  # the third submit of a context names its installed key on each engine
            hs = [P.aes_ctr_submit(ctx, icbs[0], src0.data_ptr(), dst0.data_ptr(), n),
                  P.aes_ctr_submit(ctx, icbs[1], src1.data_ptr(), dst1.data_ptr(), n),
                  P.aes_ctr_submit(ctx, icbs[2], hsrc, hdst_a, n),     # host -> host: the engines in turn
                  P.aes_ctr_submit(ctx, icbs[2], hsrc, hdst_b, n)]
            assert hs[0] >> 56 == 0 and hs[1] >> 56 == 1
            assert {hs[2] >> 56, hs[3] >> 56} == {0, 1}
            _wait_all(P, hs)
            assert G.first_mismatch(dst0.cpu().numpy(), o.ctr(key, icbs[0], data[0])) == -1
            assert G.first_mismatch(dst1.cpu().numpy(), o.ctr(key, icbs[1], data[1])) == -1
            want = o.ctr(key, icbs[2], data[2])
            assert G.first_mismatch(P.host_view(hdst_a, n).copy(), want) == -1
            assert G.first_mismatch(P.host_view(hdst_b, n).copy(), want) == -1
        with pytest.raises(P.AesOffError) as e:  # src on GPU 0, dst on GPU 1: nobody can reach both
            P.aes_ctr_submit(ctx, icbs[0], src0.data_ptr(), dst1.data_ptr(), n)
        assert e.value.code == P.AES_E_INVAL
        P.aes_engine_stop_device(1)
        with pytest.raises(P.AesOffError) as e:  # GPU 1's memory, and GPU 1 runs no engine any more
            P.aes_ctr_submit(ctx, icbs[1], src1.data_ptr(), dst1.data_ptr(), n)
        assert e.value.code == P.AES_E_STOPPED
        h = P.aes_ctr_submit(ctx, icbs[3], src0.data_ptr(), dst0.data_ptr(), n)  # engine 0 keeps serving
        _wait_all(P, [h])
        assert G.first_mismatch(dst0.cpu().numpy(), o.ctr(key, icbs[3], data[0])) == -1
    finally:
        P.aes_engine_stop()
        for p in (hsrc, hdst_a, hdst_b):
            P.aes_host_free(p)
        P.aes_ctx_destroy(ctx)

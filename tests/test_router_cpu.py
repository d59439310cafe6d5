"""-m "not gpu": the request router of the multi-GPU path (csrc/aesoff_router.cpp).
One engine per GPU, no exchange step: a request runs where its dst lives, else where its src lives; requests
between host buffers go round the running engines; memory of a GPU without an engine is refused.  The owner
look-up is remembered per 2 MiB page (tested here over a synthetic address map; on a GPU box the resolver is
cudaPointerGetAttributes)."""
import ctypes

import numpy as np

import paper_2607_02630_b200.binding as B

HOST = -2
L = B._lib
L.aesoff_test_route_decide.restype = ctypes.c_int
L.aesoff_test_route_decide.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_uint32, ctypes.c_void_p]
L.aesoff_test_route_many.restype = ctypes.c_uint64
L.aesoff_test_route_many.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_uint32, ctypes.c_void_p, ctypes.c_int]


def decide(src, dst, mask, rr):
    return L.aesoff_test_route_decide(src, dst, mask, ctypes.byref(rr))


def test_device_memory_decides_and_two_owners_are_refused():
    rr = ctypes.c_uint32(0)
    assert decide(3, 5, 0xFF, rr) == -2         # src on GPU 3, dst on GPU 5: no engine reaches both (AES_E_INVAL)
    assert decide(5, 5, 0xFF, rr) == 5
    assert decide(3, HOST, 0xFF, rr) == 3       # host dst: src decides
    assert decide(HOST, 6, 0xFF, rr) == 6
    assert rr.value == 0                        # no round-robin turn was spent on them


def test_owner_without_engine_is_refused_not_rerouted():
    rr = ctypes.c_uint32(0)
    assert decide(HOST, 2, 0b0011, rr) == -1    # the payload lives on GPU 2, which runs no engine
    assert decide(2, HOST, 0b0011, rr) == -1
    assert decide(1, 1, 0, rr) == -1            # nothing runs


def test_host_to_host_requests_go_round_the_running_engines():
    rr = ctypes.c_uint32(0)
    mask = 0b10110010                           # engines on GPUs 1, 4, 5, 7
    got = [decide(HOST, HOST, mask, rr) for _ in range(12)]
    assert got == [1, 4, 5, 7] * 3
    assert rr.value == 12
    rr = ctypes.c_uint32(0)
    assert [decide(HOST, HOST, 0b100, rr) for _ in range(3)] == [2, 2, 2]


def _dev_addr(dev, off):
    return (1 << 40) | (dev << 30) | off


def test_routes_over_a_synthetic_address_map_and_the_page_cache():
    rng = np.random.Generator(np.random.Philox(key=[260702630, 9100]))
    n = 5000
    dev = rng.integers(0, 8, size=n)
    # each device's requests reuse a pool of 4 pages (2 MiB each): 32 pages in all fit the 64-entry cache
    page = rng.integers(0, 4, size=n)
    off = rng.integers(0, 1 << 17, size=n) * 16
    dsts = np.asarray([_dev_addr(int(d), int(p) * (1 << 21) + int(o)) for d, p, o in zip(dev, page, off)], dtype=np.uint64)
    srcs = np.asarray([_dev_addr(int(d), int(p) * (1 << 21)) for d, p in zip(dev, page)], dtype=np.uint64)  # same page, same owner
    out = np.zeros(n, dtype=np.int32)
    calls = L.aesoff_test_route_many(srcs.ctypes.data, dsts.ctypes.data, n, 0xFF, out.ctypes.data, 1)
    assert (out == dev).all()
    assert calls <= 64, "owners are remembered per 2 MiB page: %d look-ups for %d requests over 32 pages" % (calls, n)
    # second pass: everything is remembered (a few pages may have evicted one another in the direct-mapped cache)
    calls2 = L.aesoff_test_route_many(srcs.ctypes.data, dsts.ctypes.data, n, 0xFF, out.ctypes.data, 0)
    assert calls2 <= calls and (out == dev).all()
    # after a flush every page is asked for again
    calls3 = L.aesoff_test_route_many(srcs.ctypes.data, dsts.ctypes.data, n, 0xFF, out.ctypes.data, 1)
    assert calls3 >= 32
    # engines on GPUs 0..3 only: requests for 4..7 are refused, the others unchanged
    L.aesoff_test_route_many(srcs.ctypes.data, dsts.ctypes.data, n, 0x0F, out.ctypes.data, 0)
    assert (out[dev < 4] == dev[dev < 4]).all() and (out[dev >= 4] == -1).all()


def test_host_buffers_mixed_with_device_buffers():
    host = np.asarray([0x5E0000001000 + 4096 * i for i in range(8)], dtype=np.uint64)  # bit 40 clear: host memory in the synthetic map
    dsts = host.copy()
    srcs = host.copy()
    srcs[3] = _dev_addr(6, 64)                  # device src, host dst: GPU 6
    dsts[5] = _dev_addr(2, 128)                 # host src, device dst: GPU 2
    out = np.zeros(8, dtype=np.int32)
    L.aesoff_test_route_many(srcs.ctypes.data, dsts.ctypes.data, 8, 0b01000101, out.ctypes.data, 1)  # engines on 0, 2, 6
    assert out[3] == 6 and out[5] == 2
    rest = [int(out[i]) for i in range(8) if i not in (3, 5)]
    assert rest == [0, 2, 6, 0, 2, 6]
    # src on GPU 0, dst on GPU 2, both with an engine: refused (-2 -> AES_E_INVAL), whichever is looked at first
    srcs[1], dsts[1] = _dev_addr(0, 256), _dev_addr(2, 512)
    L.aesoff_test_route_many(srcs.ctypes.data, dsts.ctypes.data, 8, 0b01000101, out.ctypes.data, 1)
    assert out[1] == -2 and out[3] == 6 and out[5] == 2


def test_handles_name_their_engine_and_bad_ones_are_invalid():
    # top byte = device index: a handle of an engine that does not exist is AES_E_INVAL, never a crash
    assert L.aes_poll(ctypes.c_uint64((9 << 56) | 1)) == B.AES_E_INVAL
    assert L.aes_poll(ctypes.c_uint64((3 << 56) | 12345)) == B.AES_E_INVAL   # engine 3 never issued it
    assert L.aes_poll(ctypes.c_uint64(0)) == B.AES_E_INVAL
    import pytest
    with pytest.raises(B.AesOffError) as e:
        B.aes_engine_stop_device(1)
    assert e.value.code == B.AES_E_STOPPED
    assert B.aes_engine_info(5)["running"] == 0 and B.aes_engine_info()["engines_running"] == 0

"""Thin ctypes binding of include/aesoff.h -- argument marshalling only.

Every step of the path (key expansion, submission ring, dispatch, counter blocks,
cipher, XOR/store, completion) runs inside ``libaesoff.so``; nothing here
computes.  The function names are those of the C ABI.  There is no CPU fallback:
if the shared library is missing this module raises at import, and on a machine
without a CUDA device every compute call fails with ``AES_E_CUDA``.

Pointers are plain integers (``tensor.data_ptr()`` for device memory, the address
returned by ``aes_host_alloc`` for pinned host memory).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libaesoff.so")

AES_OK = 0
AES_FINE_ROWS_OFF = 0xFFFFFFFF
AES_ENGINE_NO_DECRYPT = 1
AES_E_INVAL = -1
AES_E_KEYBITS = -2
AES_E_ALIGN = -3
AES_E_OVERLAP = -4
AES_E_AGAIN = -5
AES_E_TIMEOUT = -6
AES_E_STOPPED = -7
AES_E_CUDA = -8
AES_E_BUSY = -9
AES_E_NOMEM = -10
AES_E_TOOBIG = -11
AES_STATIC_MAX_BYTES = 64 << 20


class AesOffError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__("%s: %s (%d)" % (where, aes_strerror(code), code))


class aes_engine_opts_t(ctypes.Structure):
    _fields_ = [("ring_slots", ctypes.c_uint32), ("chunk_rows", ctypes.c_uint32), ("n_ctas", ctypes.c_uint32),
                ("idle_exit_ms", ctypes.c_uint32), ("fine_rows", ctypes.c_uint32), ("n_dispatchers", ctypes.c_uint32),
                ("flags", ctypes.c_uint32), ("reserved", ctypes.c_uint32 * 1)]


class aes_engine_info_t(ctypes.Structure):
    _fields_ = [("running", ctypes.c_int32), ("device", ctypes.c_int32), ("sm_count", ctypes.c_int32),
                ("n_ctas", ctypes.c_int32), ("threads_per_cta", ctypes.c_int32), ("worker_warps_per_cta", ctypes.c_int32),
                ("ring_slots", ctypes.c_uint32), ("chunk_rows", ctypes.c_uint32),
                ("smem_bytes_per_cta", ctypes.c_uint32), ("n_dispatchers", ctypes.c_uint32),
                ("submitted", ctypes.c_uint64), ("completed", ctypes.c_uint64), ("kernel_launches", ctypes.c_uint64),
                ("cut_eighths", ctypes.c_uint64), ("cut_halves", ctypes.c_uint64), ("cut_rows", ctypes.c_uint64),
                ("engines_running", ctypes.c_uint32), ("reserved1", ctypes.c_uint32)]


class aes_calib_t(ctypes.Structure):
    _fields_ = [("lookups_per_clk_per_sm", ctypes.c_double), ("alu_instr_per_clk_per_sm", ctypes.c_double),
                ("copy_gbs", ctypes.c_double), ("sm_mhz", ctypes.c_double), ("sm_count", ctypes.c_int32),
                ("reserved", ctypes.c_int32), ("round_lookups_per_clk_per_sm", ctypes.c_double),
                ("bitslice_sboxes_per_clk_per_sm", ctypes.c_double), ("bitslice_mismatches", ctypes.c_int32),
                ("reserved2", ctypes.c_int32)]


class aes_loop_spec_t(ctypes.Structure):
    _fields_ = [("n", ctypes.c_size_t), ("window", ctypes.c_uint32), ("repeat", ctypes.c_uint32),
                ("ctx", ctypes.c_void_p), ("keys", ctypes.c_void_p), ("keybits", ctypes.c_void_p),
                ("nonces", ctypes.c_void_p), ("srcs", ctypes.c_void_p), ("dsts", ctypes.c_void_p),
                ("lens", ctypes.c_void_p), ("mode", ctypes.c_uint32), ("reserved", ctypes.c_uint32)]


class aes_loop_result_t(ctypes.Structure):
    _fields_ = [("elapsed_ns", ctypes.c_uint64), ("bytes", ctypes.c_uint64), ("requests", ctypes.c_uint64),
                ("ring_full_spins", ctypes.c_uint64), ("max_in_flight", ctypes.c_uint64)]


def _load() -> ctypes.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "%s is missing: build it with `python -m paper_2607_02630_b200.build` "
            "(or __graft_entry__.build()).  There is no CPU fallback." % LIB_PATH)
    L = ctypes.CDLL(LIB_PATH)
    vp, u64, i32, sz = ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int, ctypes.c_size_t
    sigs = {
        "aes_engine_start": (i32, [i32, vp]),
        "aes_engine_stop": (i32, []),
        "aes_engine_info": (i32, [vp]),
        "aes_engine_info_device": (i32, [i32, vp]),
        "aes_engine_stop_device": (i32, [i32]),
        "aes_route_flush": (None, []),
        "aes_ctx_create": (vp, [vp, i32]),
        "aes_ctx_destroy": (None, [vp]),
        "aes_ctx_round_keys": (i32, [vp, vp]),
        "aes_ctr_submit": (u64, [vp, vp, vp, vp, sz]),
        "aes_ecb_submit": (u64, [vp, i32, vp, vp, sz]),
        "aes_cbc_decrypt_submit": (u64, [vp, vp, vp, vp, sz]),
        "aes_mode_launch_batch": (i32, [vp, vp, vp, vp, vp, vp, sz, i32, vp, ctypes.c_uint32]),
        "aes_poll": (i32, [u64]),
        "aes_wait": (i32, [u64, u64]),
        "aes_last_error": (i32, []),
        "aes_strerror": (ctypes.c_char_p, [i32]),
        "aes_ctr_launch_batch": (i32, [vp, vp, vp, vp, vp, sz, i32, vp, ctypes.c_uint32]),
        "aes_ctr_launch_static": (i32, [vp, vp, vp, vp, sz, i32, vp]),
        "aes_host_alloc": (vp, [sz]),
        "aes_host_free": (None, [vp]),
        "aes_host_register": (i32, [vp, sz]),
        "aes_host_unregister": (i32, [vp]),
        "aes_loop_run": (i32, [vp, vp, vp]),
        "aes_openloop_run": (i32, [vp, vp, i32, vp, vp]),
        "aes_loop_run_mt": (i32, [vp, ctypes.c_uint32, vp, vp]),
        "aes_calibrate": (i32, [i32, vp]),
    }
    for name, (res, args) in sigs.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    return L


_lib = _load()
EXPORTS = ("aes_engine_start", "aes_engine_stop", "aes_engine_info", "aes_engine_info_device", "aes_engine_stop_device", "aes_route_flush", "aes_ctx_create", "aes_ctx_destroy",
           "aes_ctx_round_keys", "aes_ctr_submit", "aes_ecb_submit", "aes_cbc_decrypt_submit", "aes_mode_launch_batch", "aes_poll", "aes_wait", "aes_last_error", "aes_strerror",
           "aes_ctr_launch_batch", "aes_ctr_launch_static", "aes_host_alloc", "aes_host_free", "aes_host_register", "aes_host_unregister", "aes_loop_run", "aes_loop_run_mt", "aes_openloop_run", "aes_calibrate")


def aes_strerror(code: int) -> str:
    return _lib.aes_strerror(code).decode()


def aes_last_error() -> int:
    return _lib.aes_last_error()


def _check(rc: int, where: str) -> None:
    if rc != AES_OK:
        raise AesOffError(rc, where)


# ---- engine ---------------------------------------------------------------------------------
def aes_engine_start(device: int = 0, ring_slots: int = 0, chunk_rows: int = 0, n_ctas: int = 0,
                     idle_exit_ms: int = 0, fine_rows: int = 0, n_dispatchers: int = 0, flags: int = 0) -> None:
    o = aes_engine_opts_t(ring_slots, chunk_rows, n_ctas, idle_exit_ms, fine_rows, n_dispatchers, flags)
    _check(_lib.aes_engine_start(device, ctypes.byref(o)), "aes_engine_start")


def aes_engine_stop() -> None:
    _check(_lib.aes_engine_stop(), "aes_engine_stop")


def aes_engine_stop_device(device: int) -> None:
    _check(_lib.aes_engine_stop_device(device), "aes_engine_stop_device")


def aes_route_flush() -> None:
    _lib.aes_route_flush()


def aes_engine_info(device: int | None = None) -> dict:
    info = aes_engine_info_t()
    if device is None:
        _check(_lib.aes_engine_info(ctypes.byref(info)), "aes_engine_info")
    else:
        _check(_lib.aes_engine_info_device(device, ctypes.byref(info)), "aes_engine_info_device")
    return {k: getattr(info, k) for k, _ in aes_engine_info_t._fields_ if k != "reserved1"}


# ---- contexts ---------------------------------------------------------------------------------
def aes_ctx_create(key: bytes, keybits: int | None = None) -> int:
    key = bytes(key)
    ctx = _lib.aes_ctx_create(key, 8 * len(key) if keybits is None else keybits)
    if not ctx:
        raise AesOffError(aes_last_error(), "aes_ctx_create")
    return ctx


def aes_ctx_destroy(ctx: int) -> None:
    _lib.aes_ctx_destroy(ctx)


def aes_ctx_round_keys(ctx: int) -> tuple:
    buf = ctypes.create_string_buffer(240)
    nr = _lib.aes_ctx_round_keys(ctx, buf)
    if nr < 0:
        raise AesOffError(nr, "aes_ctx_round_keys")
    return buf.raw[: 16 * (nr + 1)], nr


# ---- submit / completion ------------------------------------------------------------------------
def aes_ctr_submit(ctx: int, nonce: bytes, src: int, dst: int, length: int) -> int:
    """Returns the handle; raises AesOffError (code AES_E_AGAIN when the ring is full)."""
    h = _lib.aes_ctr_submit(ctx, bytes(nonce), src, dst, length)
    if h == 0:
        raise AesOffError(aes_last_error(), "aes_ctr_submit")
    return h


def aes_ecb_submit(ctx: int, decrypt: bool, src: int, dst: int, length: int) -> int:
    h = _lib.aes_ecb_submit(ctx, 1 if decrypt else 0, src, dst, length)
    if h == 0:
        raise AesOffError(aes_last_error(), "aes_ecb_submit")
    return h


def aes_cbc_decrypt_submit(ctx: int, iv: bytes, src: int, dst: int, length: int) -> int:
    h = _lib.aes_cbc_decrypt_submit(ctx, bytes(iv), src, dst, length)
    if h == 0:
        raise AesOffError(aes_last_error(), "aes_cbc_decrypt_submit")
    return h


def aes_poll(handle: int) -> bool:
    r = _lib.aes_poll(handle)
    if r < 0:
        raise AesOffError(r, "aes_poll")
    return r == 1


def aes_wait(handle: int, timeout_ns: int = 10_000_000_000) -> None:
    _check(_lib.aes_wait(handle, timeout_ns), "aes_wait")


# ---- launch backend -----------------------------------------------------------------------------
def _ptr_array(values) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(values, dtype=np.uint64))


def aes_ctr_launch_batch(ctxs, nonces, srcs, dsts, lens, device: int = 0, cuda_stream: int = 0,
                         chunk_rows: int = 0) -> None:
    """ctxs/srcs/dsts/lens: sequences of n ints; nonces: n x 16 bytes (bytes or uint8 array)."""
    n = len(lens)
    a_ctx, a_src, a_dst, a_len = _ptr_array(ctxs), _ptr_array(srcs), _ptr_array(dsts), _ptr_array(lens)
    a_non = np.ascontiguousarray(np.frombuffer(bytes(nonces), dtype=np.uint8) if isinstance(nonces, (bytes, bytearray))
                                 else np.asarray(nonces, dtype=np.uint8)).reshape(-1)
    assert a_non.size == 16 * n and a_ctx.size == n and a_src.size == n and a_dst.size == n
    _check(_lib.aes_ctr_launch_batch(a_ctx.ctypes.data, a_non.ctypes.data, a_src.ctypes.data, a_dst.ctypes.data,
                                     a_len.ctypes.data, n, device, cuda_stream, chunk_rows), "aes_ctr_launch_batch")


def aes_ctr_launch_static(ctx, nonce: bytes, src: int, dst: int, nbytes: int, device: int = 0, cuda_stream: int = 0) -> None:
    """One CTR request through the launch backend that allocates nothing (its queue is a static device array of the
    library, for callers that cannot cudaMalloc: see include/aesoff.h).  nbytes <= AES_STATIC_MAX_BYTES, else
    AES_E_TOOBIG.  Enqueues on cuda_stream and returns; the caller synchronises."""
    assert len(nonce) == 16
    _check(_lib.aes_ctr_launch_static(ctx, bytes(nonce), src, dst, nbytes, device, cuda_stream), "aes_ctr_launch_static")


AES_MODE_CTR, AES_MODE_ECB_ENC, AES_MODE_ECB_DEC, AES_MODE_CBC_DEC = 0, 1, 2, 3


def aes_mode_launch_batch(modes, ctxs, nonces, srcs, dsts, lens, device: int = 0, cuda_stream: int = 0,
                          chunk_rows: int = 0) -> None:
    """aes_ctr_launch_batch with a mode per request (AES_MODE_*); nonces: n x 16 bytes (ICB / IV / ignored)."""
    n = len(lens)
    a_mode = np.ascontiguousarray(np.asarray(modes, dtype=np.int32))
    a_ctx, a_src, a_dst, a_len = _ptr_array(ctxs), _ptr_array(srcs), _ptr_array(dsts), _ptr_array(lens)
    a_non = np.ascontiguousarray(np.frombuffer(bytes(nonces), dtype=np.uint8) if isinstance(nonces, (bytes, bytearray))
                                 else np.asarray(nonces, dtype=np.uint8)).reshape(-1)
    assert a_non.size == 16 * n and a_ctx.size == n and a_src.size == n and a_dst.size == n and a_mode.size == n
    _check(_lib.aes_mode_launch_batch(a_mode.ctypes.data, a_ctx.ctypes.data, a_non.ctypes.data, a_src.ctypes.data,
                                      a_dst.ctypes.data, a_len.ctypes.data, n, device, cuda_stream, chunk_rows),
           "aes_mode_launch_batch")


# ---- pinned host memory ---------------------------------------------------------------------------
def aes_host_alloc(nbytes: int) -> int:
    p = _lib.aes_host_alloc(nbytes)
    if not p:
        raise AesOffError(aes_last_error(), "aes_host_alloc")
    return p


def aes_host_free(ptr: int) -> None:
    _lib.aes_host_free(ptr)


def aes_host_register(ptr: int, nbytes: int) -> None:
    """Page-locks caller-owned host memory in place (e.g. ``ndarray.ctypes.data``) so that it can be submitted."""
    _check(_lib.aes_host_register(ptr, nbytes), "aes_host_register")


def aes_host_unregister(ptr: int) -> None:
    _check(_lib.aes_host_unregister(ptr), "aes_host_unregister")


def host_view(ptr: int, nbytes: int) -> np.ndarray:
    """uint8 numpy view of memory returned by aes_host_alloc (no copy)."""
    return np.ctypeslib.as_array((ctypes.c_uint8 * nbytes).from_address(ptr))


# ---- closed-loop executor ---------------------------------------------------------------------------
def aes_loop_run(nonces, srcs, dsts, lens, window: int, ctx: int = 0, keys=None, keybits=None, repeat: int = 1,
                 want_latency: bool = True, threads: int = 1, mode: int = 0) -> dict:
    """Runs the native closed loop (see aes_loop_run in aesoff.h).  keys: n x 32 uint8 (16 used for
    128-bit keys) with keybits: n int32, or a shared ``ctx``.  Returns elapsed_ns, bytes, requests,
    ring_full_spins, max_in_flight and (optionally) lat_ns as a float64 array of n*repeat entries."""
    n = len(lens)
    a_src, a_dst, a_len = _ptr_array(srcs), _ptr_array(dsts), _ptr_array(lens)
    a_non = np.ascontiguousarray(np.asarray(nonces, dtype=np.uint8)).reshape(-1)
    assert a_non.size == 16 * n
    spec = aes_loop_spec_t()
    spec.n, spec.window, spec.repeat = n, window, repeat
    spec.ctx = ctx or None
    spec.mode = mode
    keep = []
    if keys is not None:
        a_keys = np.ascontiguousarray(np.asarray(keys, dtype=np.uint8)).reshape(-1)
        a_kb = np.ascontiguousarray(np.asarray(keybits, dtype=np.int32))
        assert a_keys.size == 32 * n and a_kb.size == n
        spec.keys, spec.keybits = a_keys.ctypes.data, a_kb.ctypes.data
        keep += [a_keys, a_kb]
    spec.nonces, spec.srcs, spec.dsts, spec.lens = a_non.ctypes.data, a_src.ctypes.data, a_dst.ctypes.data, a_len.ctypes.data
    res = aes_loop_result_t()
    lat = np.zeros(n * repeat, dtype=np.float64) if want_latency else None
    if threads > 1:
        _check(_lib.aes_loop_run_mt(ctypes.byref(spec), threads, ctypes.byref(res), lat.ctypes.data if lat is not None else None),
               "aes_loop_run_mt")
    else:
        _check(_lib.aes_loop_run(ctypes.byref(spec), ctypes.byref(res), lat.ctypes.data if lat is not None else None),
               "aes_loop_run")
    out = {k: getattr(res, k) for k, _ in aes_loop_result_t._fields_}
    out["lat_ns"] = lat
    return out


def aes_loop_prepare(nonces, srcs, dsts, lens, window: int, ctx: int, repeat: int = 1, mode: int = 0):
    """Marshals a closed-loop run over a shared context ONCE and returns a function that runs it (aes_loop_run in
    aesoff.h) and returns (elapsed_ns, bytes, requests): for callers that repeat the same batch, e.g. bench.py's timed
    steps, so that no per-step Python marshalling sits inside a timed region.  The arrays are kept alive by the closure."""
    n = len(lens)
    a_src, a_dst, a_len = _ptr_array(srcs), _ptr_array(dsts), _ptr_array(lens)
    a_non = np.ascontiguousarray(np.asarray(nonces, dtype=np.uint8)).reshape(-1)
    assert a_non.size == 16 * n
    spec = aes_loop_spec_t()
    spec.n, spec.window, spec.repeat, spec.ctx, spec.mode = n, window, repeat, ctx, mode
    spec.nonces, spec.srcs, spec.dsts, spec.lens = a_non.ctypes.data, a_src.ctypes.data, a_dst.ctypes.data, a_len.ctypes.data
    res = aes_loop_result_t()
    p_spec, p_res, run = ctypes.byref(spec), ctypes.byref(res), _lib.aes_loop_run
    keep = (a_src, a_dst, a_len, a_non, spec, res)

    def go():
        rc = run(p_spec, p_res, None)
        if rc != AES_OK:
            raise AesOffError(rc, "aes_loop_run")
        return res.elapsed_ns, res.bytes, res.requests

    go.keep = keep
    return go


def aes_openloop_run(nonces, srcs, dsts, lens, arrival_ns, ctx: int, blocking: bool = False) -> dict:
    """Runs the native open loop (see aes_openloop_run in aesoff.h): request i is submitted once
    arrival_ns[i] has passed.  Returns elapsed_ns, bytes, requests, ring_full_spins, max_in_flight, lat_ns."""
    n = len(lens)
    a_src, a_dst, a_len = _ptr_array(srcs), _ptr_array(dsts), _ptr_array(lens)
    a_non = np.ascontiguousarray(np.asarray(nonces, dtype=np.uint8)).reshape(-1)
    a_arr = np.ascontiguousarray(np.asarray(arrival_ns, dtype=np.uint64))
    assert a_non.size == 16 * n and a_arr.size == n
    spec = aes_loop_spec_t()
    spec.n, spec.window, spec.repeat = n, 0, 1
    spec.ctx = ctx
    spec.nonces, spec.srcs, spec.dsts, spec.lens = a_non.ctypes.data, a_src.ctypes.data, a_dst.ctypes.data, a_len.ctypes.data
    res = aes_loop_result_t()
    lat = np.zeros(n, dtype=np.float64)
    _check(_lib.aes_openloop_run(ctypes.byref(spec), a_arr.ctypes.data, 1 if blocking else 0, ctypes.byref(res),
                                 lat.ctypes.data), "aes_openloop_run")
    out = {k: getattr(res, k) for k, _ in aes_loop_result_t._fields_}
    out["lat_ns"] = lat
    return out


def aes_calibrate(device: int = 0) -> dict:
    """Calibration microkernels (see aes_calibrate in aesoff.h)."""
    c = aes_calib_t()
    _check(_lib.aes_calibrate(device, ctypes.byref(c)), "aes_calibrate")
    return {k: getattr(c, k) for k, _ in aes_calib_t._fields_ if not k.startswith("reserved")}

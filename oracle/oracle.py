"""ctypes loader for oracle/aes_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It imports nothing from
``paper_2607_02630_b200`` (the CUDA path) and that package imports nothing
from here.  ``build()`` compiles the C oracle with gcc; building the checker is
not using it.

The functions mirror aes_oracle.h (which cites FIPS-197 / SP 800-38A section by
section); this file only marshals bytes in and out.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "aes_oracle.c")
_HDR = os.path.join(_HERE, "aes_oracle.h")
_OUT_DIR = os.path.join(_HERE, "build")
_SO = os.path.join(_OUT_DIR, "libaes_oracle.so")

_lib = None
_lock = threading.Lock()

_u8p = ctypes.POINTER(ctypes.c_uint8)


def build(force: bool = False) -> str:
    """Compile aes_oracle.c -> oracle/build/libaes_oracle.so (plain gcc -O2)."""
    os.makedirs(_OUT_DIR, exist_ok=True)
    stale = (
        force
        or not os.path.exists(_SO)
        or os.path.getmtime(_SO) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    )
    if stale:
        tmp = _SO + ".%d.tmp" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-Wall", "-Wextra", "-shared", "-fPIC", "-o", tmp, _SRC]
        )
        os.replace(tmp, _SO)
    return _SO


def lib() -> ctypes.CDLL:
    global _lib
    with _lock:
        if _lib is None:
            L = ctypes.CDLL(build())
            u8, i32, u64, sz = ctypes.c_uint8, ctypes.c_int, ctypes.c_uint64, ctypes.c_size_t
            for name, res, args in [
                ("oracle_xtime", u8, [u8]),
                ("oracle_gf_mul", u8, [u8, u8]),
                ("oracle_gf_inv", u8, [u8]),
                ("oracle_sbox", u8, [u8]),
                ("oracle_inv_sbox", u8, [u8]),
                ("oracle_rcon", u8, [i32]),
                ("oracle_sub_bytes", None, [ctypes.c_void_p]),
                ("oracle_shift_rows", None, [ctypes.c_void_p]),
                ("oracle_mix_columns", None, [ctypes.c_void_p]),
                ("oracle_add_round_key", None, [ctypes.c_void_p, ctypes.c_void_p]),
                ("oracle_inv_sub_bytes", None, [ctypes.c_void_p]),
                ("oracle_inv_shift_rows", None, [ctypes.c_void_p]),
                ("oracle_inv_mix_columns", None, [ctypes.c_void_p]),
                ("oracle_key_expand", i32, [ctypes.c_void_p, i32, ctypes.c_void_p]),
                ("oracle_encrypt_block", None, [ctypes.c_void_p, i32, ctypes.c_void_p, ctypes.c_void_p]),
                ("oracle_decrypt_block", None, [ctypes.c_void_p, i32, ctypes.c_void_p, ctypes.c_void_p]),
                ("oracle_ctr", None, [ctypes.c_void_p, i32, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, sz]),
                ("oracle_ctr_at", None, [ctypes.c_void_p, i32, ctypes.c_void_p, u64, ctypes.c_void_p, ctypes.c_void_p, sz]),
                ("oracle_ctr_add", None, [ctypes.c_void_p, u64, ctypes.c_void_p]),
                ("oracle_ecb_encrypt", None, [ctypes.c_void_p, i32, ctypes.c_void_p, ctypes.c_void_p, sz]),
                ("oracle_ecb_decrypt", None, [ctypes.c_void_p, i32, ctypes.c_void_p, ctypes.c_void_p, sz]),
                ("oracle_cbc_encrypt", None, [ctypes.c_void_p, i32, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, sz]),
                ("oracle_cbc_decrypt", None, [ctypes.c_void_p, i32, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, sz]),
            ]:
                fn = getattr(L, name)
                fn.restype = res
                fn.argtypes = args
            _lib = L
    return _lib


# ---------------------------------------------------------------------------
# byte-level helpers
# ---------------------------------------------------------------------------
def _state_op(name: str, state: bytes, *extra: bytes) -> bytes:
    assert len(state) == 16
    buf = ctypes.create_string_buffer(bytes(state), 16)
    args = [ctypes.create_string_buffer(bytes(e), len(e)) for e in extra]
    getattr(lib(), name)(buf, *args)
    return buf.raw


def sub_bytes(s): return _state_op("oracle_sub_bytes", s)
def shift_rows(s): return _state_op("oracle_shift_rows", s)
def mix_columns(s): return _state_op("oracle_mix_columns", s)
def add_round_key(s, rk16): return _state_op("oracle_add_round_key", s, rk16)
def inv_sub_bytes(s): return _state_op("oracle_inv_sub_bytes", s)
def inv_shift_rows(s): return _state_op("oracle_inv_shift_rows", s)
def inv_mix_columns(s): return _state_op("oracle_inv_mix_columns", s)


def key_expand(key: bytes) -> tuple[bytes, int]:
    """-> (round keys, Nr); raises ValueError for a key that is not 16/24/32 bytes."""
    keybits = 8 * len(key)
    rk = ctypes.create_string_buffer(240)
    nr = lib().oracle_key_expand(bytes(key), keybits, rk)
    if nr < 0:
        raise ValueError("keybits must be 128, 192 or 256")
    return rk.raw[: 16 * (nr + 1)], nr


def encrypt_block(key: bytes, block: bytes) -> bytes:
    rk, nr = key_expand(key)
    out = ctypes.create_string_buffer(16)
    lib().oracle_encrypt_block(rk, nr, bytes(block), out)
    return out.raw


def decrypt_block(key: bytes, block: bytes) -> bytes:
    rk, nr = key_expand(key)
    out = ctypes.create_string_buffer(16)
    lib().oracle_decrypt_block(rk, nr, bytes(block), out)
    return out.raw


def ctr_add(icb: bytes, add: int) -> bytes:
    out = ctypes.create_string_buffer(16)
    lib().oracle_ctr_add(bytes(icb), add, out)
    return out.raw


def ctr(key: bytes, icb: bytes, data, block_offset: int = 0) -> bytes:
    """AES-CTR of ``data`` (bytes-like or a C-contiguous uint8 numpy array).

    ``block_offset`` starts the counter at icb + block_offset (oracle_ctr_at).
    """
    assert len(icb) == 16
    rk, nr = key_expand(key)
    mv = memoryview(data).cast("B")
    n = mv.nbytes
    out = ctypes.create_string_buffer(n) if n else ctypes.create_string_buffer(1)
    src = (ctypes.c_uint8 * n).from_buffer_copy(mv) if n else None
    lib().oracle_ctr_at(rk, nr, bytes(icb), block_offset, src, out, n)
    return out.raw[:n]


def ctr_into(key: bytes, icb: bytes, src_addr: int, dst_addr: int, n: int, block_offset: int = 0) -> None:
    """Pointer form for the timed cpu_baseline leg (no copies; releases the GIL)."""
    rk, nr = key_expand(key)
    lib().oracle_ctr_at(rk, nr, bytes(icb), block_offset, src_addr, dst_addr, n)


def _blocks(name: str, key: bytes, data, iv: bytes | None = None) -> bytes:
    rk, nr = key_expand(key)
    mv = memoryview(data).cast("B")
    n = mv.nbytes
    if n % 16:
        raise ValueError("ECB/CBC take whole 16-byte blocks (SP 800-38A sec. 6.1, 6.2)")
    out = ctypes.create_string_buffer(max(n, 1))
    src = (ctypes.c_uint8 * n).from_buffer_copy(mv) if n else None
    if iv is None:
        getattr(lib(), name)(rk, nr, src, out, n // 16)
    else:
        assert len(iv) == 16
        getattr(lib(), name)(rk, nr, bytes(iv), src, out, n // 16)
    return out.raw[:n]


def ecb_encrypt(key: bytes, data) -> bytes: return _blocks("oracle_ecb_encrypt", key, data)
def ecb_decrypt(key: bytes, data) -> bytes: return _blocks("oracle_ecb_decrypt", key, data)
def cbc_encrypt(key: bytes, iv: bytes, data) -> bytes: return _blocks("oracle_cbc_encrypt", key, data, iv)
def cbc_decrypt(key: bytes, iv: bytes, data) -> bytes: return _blocks("oracle_cbc_decrypt", key, data, iv)

"""Pins of the oracle's ECB and CBC functions (SP 800-38A sec. 6.1, 6.2) against things
other than the oracle:

M1  the values PRINTED in SP 800-38A Appendix F.1 (ECB) and F.2 (CBC), AES-128/192/256, both directions
    (tests/golden/sp800_38a_f1_f2_ecb_cbc.txt)
M2  library routines on seeded random keys / IVs / lengths: Python `cryptography` and the system libcrypto
    through its EVP C API (decryption contexts: EVP_DecryptInit_ex), lengths 0 .. 64 KiB + 16
M3  structure that a plausible mistake breaks: a flipped ciphertext bit garbles exactly its own block and flips
    exactly that bit in the next one (CBC decryption, sec. 6.2 / appendix D); equal ciphertext blocks decrypt to
    equal blocks in ECB and not in CBC; a window [a, b) decrypts alone with IV = C_{a-1} (what GPU chunking of
    CBC decryption relies on); in place == out of place
"""
import ctypes
import ctypes.util

import numpy as np
import pytest

from oracle import oracle as o
from paper_2607_02630_b200 import workloads

cryptography = pytest.importorskip("cryptography")
from cryptography.hazmat.primitives.ciphers import Cipher, algorithms, modes  # noqa: E402

RNG = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 78]))
LENS = (0, 16, 32, 48, 4096, 4112, 65536 + 16)


def _lib(mode, key, data, decrypt):
    c = Cipher(algorithms.AES(key), mode)
    x = c.decryptor() if decrypt else c.encryptor()
    return x.update(bytes(data)) + x.finalize()


# --- M1 ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("tag,key", [("f11", "k128"), ("f13", "k192"), ("f15", "k256")])
def test_sp800_38a_f1_ecb_vectors(golden, tag, key):
    g = golden("sp800_38a_f1_f2_ecb_cbc.txt")
    pt, ct = g["f.plaintext"], g[tag + ".ciphertext"]
    assert o.ecb_encrypt(g[key], pt) == ct            # F.1.1 / F.1.3 / F.1.5
    assert o.ecb_decrypt(g[key], ct) == pt            # F.1.2 / F.1.4 / F.1.6
    for j in range(4):                                # every block on its own
        assert o.ecb_decrypt(g[key], ct[16 * j:16 * j + 16]) == pt[16 * j:16 * j + 16]


@pytest.mark.parametrize("tag,key", [("f21", "k128"), ("f23", "k192"), ("f25", "k256")])
def test_sp800_38a_f2_cbc_vectors(golden, tag, key):
    g = golden("sp800_38a_f1_f2_ecb_cbc.txt")
    pt, ct, iv = g["f.plaintext"], g[tag + ".ciphertext"], g["f2.iv"]
    assert o.cbc_encrypt(g[key], iv, pt) == ct        # F.2.1 / F.2.3 / F.2.5
    assert o.cbc_decrypt(g[key], iv, ct) == pt        # F.2.2 / F.2.4 / F.2.6
    for n in (1, 2, 3):                               # prefixes: CBC is causal
        assert o.cbc_encrypt(g[key], iv, pt[:16 * n]) == ct[:16 * n]
        assert o.cbc_decrypt(g[key], iv, ct[:16 * n]) == pt[:16 * n]


def test_sp800_38a_f21_input_block(golden):
    """F.2.1 prints the cipher's "Input Block" #2 = P_2 xor C_1: the chaining feeds the PREVIOUS CIPHERTEXT block."""
    g = golden("sp800_38a_f1_f2_ecb_cbc.txt")
    ct = g["f21.ciphertext"]
    assert o.decrypt_block(g["k128"], ct[16:32]) == g["f21.input_block2"]
    x = bytes(a ^ b for a, b in zip(g["f21.input_block2"], ct[:16]))
    assert x == g["f.plaintext"][16:32]


# --- M2 ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("keylen", [16, 24, 32])
def test_m2_cryptography_ecb_cbc(keylen):
    for n in LENS:
        key, iv, data = RNG.bytes(keylen), RNG.bytes(16), RNG.bytes(n)
        assert o.ecb_encrypt(key, data) == _lib(modes.ECB(), key, data, False)
        assert o.ecb_decrypt(key, data) == _lib(modes.ECB(), key, data, True)
        assert o.cbc_encrypt(key, iv, data) == _lib(modes.CBC(iv), key, data, False)
        assert o.cbc_decrypt(key, iv, data) == _lib(modes.CBC(iv), key, data, True)


class _EvpDec:
    """System libcrypto (a separate build from the `cryptography` wheel), decryption contexts, no padding."""

    def __init__(self):
        name = ctypes.util.find_library("crypto")
        if not name:
            pytest.skip("libcrypto not found")
        L = ctypes.CDLL(name)
        L.EVP_CIPHER_CTX_new.restype = ctypes.c_void_p
        L.EVP_CIPHER_CTX_free.argtypes = [ctypes.c_void_p]
        for m in ("ecb", "cbc"):
            for b in (128, 192, 256):
                getattr(L, "EVP_aes_%d_%s" % (b, m)).restype = ctypes.c_void_p
        for f in ("EVP_DecryptInit_ex", "EVP_EncryptInit_ex"):
            getattr(L, f).argtypes = [ctypes.c_void_p] * 3 + [ctypes.c_char_p, ctypes.c_char_p]
        for f in ("EVP_DecryptUpdate", "EVP_EncryptUpdate"):
            getattr(L, f).argtypes = [ctypes.c_void_p, ctypes.c_char_p, ctypes.POINTER(ctypes.c_int), ctypes.c_char_p,
                                      ctypes.c_int]
        L.EVP_CIPHER_CTX_set_padding.argtypes = [ctypes.c_void_p, ctypes.c_int]
        self.L = L

    def run(self, mode, key, iv, data, decrypt):
        L = self.L
        ctx = L.EVP_CIPHER_CTX_new()
        try:
            ciph = getattr(L, "EVP_aes_%d_%s" % (8 * len(key), mode))()
            init, upd = (L.EVP_DecryptInit_ex, L.EVP_DecryptUpdate) if decrypt else (L.EVP_EncryptInit_ex, L.EVP_EncryptUpdate)
            assert init(ctx, ciph, None, key, iv) == 1
            L.EVP_CIPHER_CTX_set_padding(ctx, 0)
            out = ctypes.create_string_buffer(len(data) + 32)
            n = ctypes.c_int(0)
            assert upd(ctx, out, ctypes.byref(n), bytes(data), len(data)) == 1
            return out.raw[: n.value]
        finally:
            L.EVP_CIPHER_CTX_free(ctx)


@pytest.mark.parametrize("keylen", [16, 24, 32])
def test_m2_libcrypto_evp_ecb_cbc(keylen):
    evp = _EvpDec()
    for n in (16, 160, 4096, 65536 + 16):
        key, iv, data = RNG.bytes(keylen), RNG.bytes(16), RNG.bytes(n)
        assert o.ecb_decrypt(key, data) == evp.run("ecb", key, None, data, True)
        assert o.ecb_encrypt(key, data) == evp.run("ecb", key, None, data, False)
        assert o.cbc_decrypt(key, iv, data) == evp.run("cbc", key, iv, data, True)
        assert o.cbc_encrypt(key, iv, data) == evp.run("cbc", key, iv, data, False)


# --- M3 ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("keylen", [16, 32])
def test_m3_round_trips_and_rejects_partial_blocks(keylen):
    key, iv, data = RNG.bytes(keylen), RNG.bytes(16), RNG.bytes(16 * 37)
    assert o.ecb_decrypt(key, o.ecb_encrypt(key, data)) == data
    assert o.cbc_decrypt(key, iv, o.cbc_encrypt(key, iv, data)) == data
    with pytest.raises(ValueError):
        o.ecb_encrypt(key, data[:17])
    with pytest.raises(ValueError):
        o.cbc_decrypt(key, iv, data[:15])


def test_m3_cbc_error_propagation_appendix_d():
    """SP 800-38A appendix D: in CBC decryption a bit error in ciphertext block j garbles plaintext block j and
    flips the same bit of block j + 1, and nothing else."""
    key, iv = RNG.bytes(16), RNG.bytes(16)
    ct = bytearray(RNG.bytes(16 * 8))
    good = o.cbc_decrypt(key, iv, bytes(ct))
    j, bit = 3, 0x10
    ct[16 * j + 5] ^= bit
    bad = o.cbc_decrypt(key, iv, bytes(ct))
    assert bad[:16 * j] == good[:16 * j] and bad[16 * (j + 2):] == good[16 * (j + 2):]
    assert bad[16 * j:16 * j + 16] != good[16 * j:16 * j + 16]
    nxt = bytearray(good[16 * (j + 1):16 * (j + 2)])
    nxt[5] ^= bit
    assert bad[16 * (j + 1):16 * (j + 2)] == bytes(nxt)


def test_m3_equal_blocks_and_iv():
    key, iv = RNG.bytes(32), RNG.bytes(16)
    blk = RNG.bytes(16)
    pe = o.ecb_decrypt(key, blk * 4)
    assert pe[:16] == pe[16:32] == pe[32:48] == pe[48:]          # ECB: equal in, equal out
    pc = o.cbc_decrypt(key, iv, blk * 4)
    assert pc[16:32] == pc[32:48] == pc[48:] and pc[:16] != pc[16:32]  # CBC: block 1 sees the IV, the rest C_{j-1} = blk
    assert o.cbc_decrypt(key, bytes(16), blk) == o.ecb_decrypt(key, blk)  # IV = 0, one block: CBC is ECB
    # a different IV changes the first plaintext block only
    pd = o.cbc_decrypt(key, RNG.bytes(16), blk * 4)
    assert pd[16:] == pc[16:] and pd[:16] != pc[:16]


@pytest.mark.parametrize("keylen", [16, 24, 32])
def test_m3_cbc_window_decrypts_alone(keylen):
    """Blocks [a, b) of a CBC ciphertext decrypt on their own with IV = C_{a-1} (IV itself for a = 0): the property
    the GPU's chunking of CBC decryption rests on."""
    key, iv = RNG.bytes(keylen), RNG.bytes(16)
    ct = RNG.bytes(16 * 300)
    whole = o.cbc_decrypt(key, iv, ct)
    for a, b in ((0, 1), (0, 256), (1, 2), (255, 257), (256, 300), (299, 300)):
        prev = iv if a == 0 else ct[16 * (a - 1):16 * a]
        assert o.cbc_decrypt(key, prev, ct[16 * a:16 * b]) == whole[16 * a:16 * b]


def test_m3_in_place_equals_out_of_place():
    key, iv = RNG.bytes(16), RNG.bytes(16)
    data = RNG.bytes(16 * 50)
    rk, nr = o.key_expand(key)
    L = o.lib()
    for name, with_iv in (("oracle_ecb_encrypt", False), ("oracle_ecb_decrypt", False), ("oracle_cbc_encrypt", True),
                          ("oracle_cbc_decrypt", True)):
        buf = ctypes.create_string_buffer(data, len(data))
        out = ctypes.create_string_buffer(len(data))
        src = ctypes.create_string_buffer(data, len(data))
        args = (rk, nr, iv) if with_iv else (rk, nr)
        getattr(L, name)(*args, src, out, len(data) // 16)
        getattr(L, name)(*args, buf, buf, len(data) // 16)
        assert buf.raw == out.raw, name

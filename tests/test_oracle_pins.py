"""Pins P2-P10: the oracle against things other than itself.

P2  library routines: Python `cryptography` (bundled OpenSSL) and the system
    libcrypto.so.3 through its EVP C API (a separate build), ECB and CTR
P3  closed forms computable by hand from FIPS-197 sec. 4.2 / 5.1.1 / 5.2
P4  S-box invariants          P5  linear-layer invariants
P6  InvCipher(Cipher(x)) = x  P7  key schedule run backwards recovers the key
P8  CTR structure             P9  host AES-NI single rounds (hardware)
P10 brute force over one input byte vs the library
"""
import ctypes
import ctypes.util
import os
import subprocess

import numpy as np
import pytest

from oracle import oracle as o
from paper_2607_02630_b200 import workloads

cryptography = pytest.importorskip("cryptography")
from cryptography.hazmat.primitives.ciphers import Cipher, algorithms, modes  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
RNG = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 77]))


def rbytes(n):
    return RNG.bytes(n)


def lib_ecb(key, block):
    e = Cipher(algorithms.AES(key), modes.ECB()).encryptor()
    return e.update(block) + e.finalize()


def lib_ctr(key, icb, data):
    e = Cipher(algorithms.AES(key), modes.CTR(icb)).encryptor()
    return e.update(bytes(data)) + e.finalize()


# --- P2b: system libcrypto through EVP, independent of the wheel above -------
class _Evp:
    def __init__(self):
        name = ctypes.util.find_library("crypto")
        if not name:
            pytest.skip("libcrypto not found")
        L = ctypes.CDLL(name)
        L.EVP_CIPHER_CTX_new.restype = ctypes.c_void_p
        L.EVP_CIPHER_CTX_free.argtypes = [ctypes.c_void_p]
        for n in ("ecb", "ctr"):
            for b in (128, 192, 256):
                getattr(L, "EVP_aes_%d_%s" % (b, n)).restype = ctypes.c_void_p
        L.EVP_EncryptInit_ex.argtypes = [ctypes.c_void_p] * 3 + [ctypes.c_char_p, ctypes.c_char_p]
        L.EVP_EncryptUpdate.argtypes = [ctypes.c_void_p, ctypes.c_char_p, ctypes.POINTER(ctypes.c_int),
                                        ctypes.c_char_p, ctypes.c_int]
        L.EVP_CIPHER_CTX_set_padding.argtypes = [ctypes.c_void_p, ctypes.c_int]
        self.L = L

    def run(self, mode, key, iv, data):
        L = self.L
        ctx = L.EVP_CIPHER_CTX_new()
        try:
            ciph = getattr(L, "EVP_aes_%d_%s" % (8 * len(key), mode))()
            assert L.EVP_EncryptInit_ex(ctx, ciph, None, key, iv) == 1
            L.EVP_CIPHER_CTX_set_padding(ctx, 0)
            out = ctypes.create_string_buffer(len(data) + 32)
            n = ctypes.c_int(0)
            assert L.EVP_EncryptUpdate(ctx, out, ctypes.byref(n), bytes(data), len(data)) == 1
            return out.raw[: n.value]
        finally:
            L.EVP_CIPHER_CTX_free(ctx)


@pytest.fixture(scope="module")
def evp():
    return _Evp()


# ------------------------------------------------------------------ P2 ------
@pytest.mark.parametrize("keylen", [16, 24, 32])
def test_p2_block_cipher_equals_libraries(keylen, evp):
    for _ in range(64):
        key, blk = rbytes(keylen), rbytes(16)
        want = lib_ecb(key, blk)
        assert o.encrypt_block(key, blk) == want
        assert evp.run("ecb", key, None, blk) == want
        assert o.decrypt_block(key, want) == blk


LENGTHS = [0, 1, 15, 16, 17, 31, 32, 33, 255, 256, 257, 4095, 4096, 4097, 65536, (1 << 20) + 5]


@pytest.mark.parametrize("keylen", [16, 24, 32])
def test_p2_ctr_equals_libraries_on_seeded_random(keylen, evp):
    for n in LENGTHS:
        key, icb, data = rbytes(keylen), rbytes(16), rbytes(n)
        want = lib_ctr(key, icb, data)
        assert o.ctr(key, icb, data) == want, n
        if n <= 65536:
            assert evp.run("ctr", key, icb, data) == want, n


@pytest.mark.parametrize("keylen", [16, 32])
def test_p2_ctr_carry_is_128_bit_big_endian(keylen, evp):
    """DESIGN.md reading R4: the whole block increments, carries propagate past
    32 and 64 bits and wrap mod 2^128 -- and both libraries agree."""
    key = rbytes(keylen)
    for icb in workloads.edge_icbs():
        data = rbytes(16 * 400 + 7)  # carries at +1, +6 and +301 all inside
        want = lib_ctr(key, icb, data)
        assert o.ctr(key, icb, data) == want
        assert evp.run("ctr", key, icb, data) == want


def test_ctr_add_is_plain_integer_addition():
    for icb in workloads.edge_icbs() + [rbytes(16) for _ in range(16)]:
        for add in (0, 1, 2, 255, 256, 65535, (1 << 32) - 1, 1 << 32, (1 << 64) - 1):
            want = ((int.from_bytes(icb, "big") + add) % (1 << 128)).to_bytes(16, "big")
            assert o.ctr_add(icb, add) == want


def test_p2_openssl_cli_agrees():
    """Third opinion through a separate process: /usr/bin/openssl enc."""
    exe = "/usr/bin/openssl"
    if not os.path.exists(exe):
        pytest.skip("no openssl CLI")
    for keylen, name in ((16, "-aes-128-ctr"), (32, "-aes-256-ctr")):
        key, icb, data = rbytes(keylen), rbytes(16), rbytes(1000 + 3)
        got = subprocess.run([exe, "enc", name, "-K", key.hex(), "-iv", icb.hex()],
                             input=data, capture_output=True, check=True).stdout
        assert o.ctr(key, icb, data) == got


# ------------------------------------------------------------------ P3 ------
def test_p3_closed_forms():
    L = o.lib()
    assert L.oracle_xtime(0x80) == 0x1B and L.oracle_xtime(0x01) == 0x02 and L.oracle_xtime(0x57) == 0xAE
    # FIPS-197 sec. 4.2 worked example {57}*{83}={c1}; sec. 4.2.1 {57}*{13}={fe}
    assert L.oracle_gf_mul(0x57, 0x83) == 0xC1 and L.oracle_gf_mul(0x57, 0x13) == 0xFE
    # S(00): inverse of 0 is 0 -> affine constant; S(01): inv(1)=1 -> 1f ^ 63
    assert L.oracle_sbox(0x00) == 0x63 and L.oracle_sbox(0x01) == 0x7C
    # sec. 5.1.1 worked example: S({53}) = {ed}
    assert L.oracle_sbox(0x53) == 0xED
    # Rcon: successive doublings of 01, reduced: 01 02 04 08 10 20 40 80 1b 36
    assert [L.oracle_rcon(j) for j in range(1, 11)] == [1, 2, 4, 8, 16, 32, 64, 128, 0x1B, 0x36]


def test_p3_gf_mul_is_a_field_multiplication():
    L = o.lib()
    for a in range(256):
        assert L.oracle_gf_mul(a, 1) == a and L.oracle_gf_mul(a, 0) == 0
        assert L.oracle_gf_mul(a, 2) == L.oracle_xtime(a)
        if a:
            assert L.oracle_gf_mul(a, L.oracle_gf_inv(a)) == 1
    for _ in range(300):
        a, b, c = (int(x) for x in RNG.integers(0, 256, 3))
        assert L.oracle_gf_mul(a, b) == L.oracle_gf_mul(b, a)
        assert L.oracle_gf_mul(a, b ^ c) == L.oracle_gf_mul(a, b) ^ L.oracle_gf_mul(a, c)
        assert L.oracle_gf_mul(L.oracle_gf_mul(a, b), c) == L.oracle_gf_mul(a, L.oracle_gf_mul(b, c))


# ------------------------------------------------------------------ P4 ------
def test_p4_sbox_invariants():
    L = o.lib()
    S = [L.oracle_sbox(a) for a in range(256)]
    assert sorted(S) == list(range(256))
    for a in range(256):
        assert L.oracle_inv_sbox(S[a]) == a
        assert S[a] != a and S[a] != (a ^ 0xFF)


# ------------------------------------------------------------------ P5 ------
def test_p5_linear_layer_invariants():
    for a in range(256):
        col = bytes([a] * 16)
        assert o.mix_columns(col) == col  # 2+3+1+1 = 1 in GF(2^8)
    for _ in range(32):
        s = rbytes(16)
        m = s
        for _k in range(4):
            m = o.mix_columns(m)
        assert m == s  # the circulant has order 4
        assert o.inv_mix_columns(o.mix_columns(s)) == s
        r = s
        for _k in range(4):
            r = o.shift_rows(r)
        assert r == s
        assert o.inv_shift_rows(o.shift_rows(s)) == s
    # ShiftRows moves row r left by r: byte (r,c) comes from (r,c+r)
    s = bytes(range(16))
    t = o.shift_rows(s)
    assert t == bytes([0, 5, 10, 15, 4, 9, 14, 3, 8, 13, 2, 7, 12, 1, 6, 11])
    # MixColumns acts on each column separately and is GF(2)-linear
    a, b = rbytes(16), rbytes(16)
    xor = bytes(x ^ y for x, y in zip(a, b))
    assert o.mix_columns(xor) == bytes(x ^ y for x, y in zip(o.mix_columns(a), o.mix_columns(b)))
    one_col = bytes([0xDB, 0x13, 0x53, 0x45]) + bytes(12)
    assert o.mix_columns(one_col)[4:] == bytes(12)


# ------------------------------------------------------------------ P6 ------
@pytest.mark.parametrize("keylen", [16, 24, 32])
def test_p6_encrypt_decrypt_round_trip(keylen):
    for _ in range(64):
        key, blk = rbytes(keylen), rbytes(16)
        assert o.decrypt_block(key, o.encrypt_block(key, blk)) == blk


# ------------------------------------------------------------------ P7 ------
@pytest.mark.parametrize("keylen", [16, 24, 32])
def test_p7_key_schedule_runs_backwards_to_the_key(keylen):
    L = o.lib()
    nk = keylen // 4
    for _ in range(16):
        key = rbytes(keylen)
        rk, nr = o.key_expand(key)
        assert rk[:keylen] == key
        w = [rk[4 * i:4 * i + 4] for i in range(4 * (nr + 1))]
        # w[i-Nk] = w[i] ^ t(w[i-1]), from the top down
        for i in range(4 * (nr + 1) - 1, nk - 1, -1):
            t = w[i - 1]
            if i % nk == 0:
                t = bytes([L.oracle_sbox(t[1]) ^ L.oracle_rcon(i // nk), L.oracle_sbox(t[2]),
                           L.oracle_sbox(t[3]), L.oracle_sbox(t[0])])
            elif nk > 6 and i % nk == 4:
                t = bytes(L.oracle_sbox(x) for x in t)
            assert bytes(x ^ y for x, y in zip(w[i], t)) == w[i - nk]


def test_key_expand_rejects_other_sizes():
    with pytest.raises(ValueError):
        o.key_expand(bytes(20))


# ------------------------------------------------------------------ P8 ------
@pytest.mark.parametrize("keylen", [16, 32])
def test_p8_ctr_structure(keylen):
    key, icb = rbytes(keylen), rbytes(16)
    n = 16 * 37 + 9
    p1, p2 = rbytes(n), rbytes(n)
    c1, c2 = o.ctr(key, icb, p1), o.ctr(key, icb, p2)
    # keystream for zeros = ECB of explicit counter blocks
    ks = o.ctr(key, icb, bytes(n))
    for j in range(0, n, 16):
        assert ks[j:j + 16] == o.encrypt_block(key, o.ctr_add(icb, j // 16))[: n - j]
    assert o.ctr(key, icb, c1) == p1                                        # involution
    assert bytes(a ^ b for a, b in zip(c1, c2)) == bytes(a ^ b for a, b in zip(p1, p2))
    for m in (0, 1, 16, 100, n - 1):
        assert o.ctr(key, icb, p1[:m]) == c1[:m]                            # prefix property
    for a in (16, 160, 16 * 36):                                            # split invariance
        assert o.ctr(key, icb, p1[:a]) + o.ctr(key, icb, p1[a:], block_offset=a // 16) == c1


# ------------------------------------------------------------------ P9 ------
@pytest.fixture(scope="module")
def aesni(tmp_path_factory):
    with open("/proc/cpuinfo") as f:
        if " aes " not in f.read().replace("\n", " "):
            pytest.skip("host CPU has no AES-NI")
    so = str(tmp_path_factory.mktemp("aesni") / "aesni.so")
    subprocess.check_call(["gcc", "-O2", "-maes", "-shared", "-fPIC", "-o", so,
                           os.path.join(HERE, "helpers", "aesni_round.c")])
    return ctypes.CDLL(so)


def test_p9_single_rounds_equal_aesni_hardware(aesni):
    out = ctypes.create_string_buffer(16)
    for _ in range(64):
        s, k = rbytes(16), rbytes(16)
        aesni.aesni_enc_round(s, k, out)
        assert o.add_round_key(o.mix_columns(o.shift_rows(o.sub_bytes(s))), k) == out.raw
        aesni.aesni_enc_last_round(s, k, out)
        assert o.add_round_key(o.shift_rows(o.sub_bytes(s)), k) == out.raw


@pytest.mark.parametrize("keylen", [16, 24, 32])
def test_p9_oracle_round_keys_drive_aesni_to_the_same_ciphertext(aesni, keylen):
    out = ctypes.create_string_buffer(16)
    for _ in range(16):
        key, blk = rbytes(keylen), rbytes(16)
        rk, nr = o.key_expand(key)
        aesni.aesni_encrypt_block(rk, nr, blk, out)
        assert out.raw == o.encrypt_block(key, blk) == lib_ecb(key, blk)


# ----------------------------------------------------------------- P10 ------
@pytest.mark.parametrize("keylen", [16, 32])
def test_p10_brute_force_each_byte_position(keylen):
    key = rbytes(keylen)
    for pos in range(16):
        for v in range(0, 256, 5 if pos else 1):
            blk = bytearray(16)
            blk[pos] = v
            assert o.encrypt_block(key, bytes(blk)) == lib_ecb(key, bytes(blk))

/*
 * aesoff_keys.cpp -- host-side key expansion and the T0 table of the product library.
 *
 * Step a1 of the path: FIPS-197 sec. 5.2 KeyExpansion().  On the engine path the expansion runs on the
 * DEVICE (the raw key rides in the descriptor, key_expand<NK> in aesoff_cipher.cuh); the host copy below
 * serves aes_ctx_round_keys() (so that tests can pin the schedule on its own) and the launch backend, which
 * ships expanded keys in its one host->device blob.  This file shares nothing with oracle/: the S-box below is
 * built from discrete logarithms to the generator {03} (a different route from the oracle's
 * search for inverses), so a slip in either shows up as a parity failure.
 */
#include <stdint.h>
#include <string.h>

#include <mutex>

#include "aesoff_internal.h"

namespace {

uint8_t g_sbox[256];
uint32_t g_T0[512]; /* T0, then Td0 (equivalent inverse cipher, FIPS-197 sec. 5.3.5) */
std::once_flag g_once;

inline uint8_t mul2(uint8_t a) { return (uint8_t)((a << 1) ^ ((a & 0x80) ? 0x1b : 0)); }

void build_tables()
{
    /* powers of the generator {03}: alog[i] = {03}^i, log its inverse map */
    uint8_t alog[256], lg[256];
    uint8_t x = 1;
    for (int i = 0; i < 255; ++i) {
        alog[i] = x;
        lg[x] = (uint8_t)i;
        x = (uint8_t)(x ^ mul2(x)); /* x * {03} */
    }
    alog[255] = alog[0];
    for (int a = 0; a < 256; ++a) {
        const uint8_t inv = a ? alog[(255 - lg[a]) % 255] : 0;
        /* affine map of sec. 5.1.1: b_i ^ b_{i+4} ^ b_{i+5} ^ b_{i+6} ^ b_{i+7} ^ c_i, c = {63} */
        uint8_t s = 0;
        for (int i = 0; i < 8; ++i) {
            const int bit = ((inv >> i) ^ (inv >> ((i + 4) & 7)) ^ (inv >> ((i + 5) & 7)) ^ (inv >> ((i + 6) & 7)) ^
                             (inv >> ((i + 7) & 7)) ^ (0x63 >> i)) & 1;
            s |= (uint8_t)(bit << i);
        }
        g_sbox[a] = s;
    }
    for (int a = 0; a < 256; ++a) {
        const uint8_t s = g_sbox[a], s2 = mul2(s), s3 = (uint8_t)(s2 ^ s);
        /* column (02,01,01,03)^T of MixColumns applied to S[a]; byte 0 of the word = row 0 */
        g_T0[a] = (uint32_t)s2 | ((uint32_t)s << 8) | ((uint32_t)s << 16) | ((uint32_t)s3 << 24);
    }
    /* Td0[x] = column (0e,09,0d,0b)^T of InvMixColumns (sec. 5.3.3) applied to InvSubBytes(x); products through the
     * same logarithms.  The four bytes of an entry xor to InvSubBytes(x) itself (0e ^ 09 ^ 0d ^ 0b = 01), which is how
     * the kernel's final round reads the inverse S-box out of this one table.                                       */
    for (int a = 0; a < 256; ++a) {
        const uint8_t x = g_sbox[a]; /* InvSubBytes(x) == a */
        auto mul = [&](uint8_t c) -> uint32_t { return a ? alog[(lg[(uint8_t)a] + lg[c]) % 255] : 0u; };
        g_T0[256 + x] = mul(0x0e) | (mul(0x09) << 8) | (mul(0x0d) << 16) | (mul(0x0b) << 24);
    }
}

inline uint32_t sub_word(uint32_t w)
{
    return (uint32_t)g_sbox[w & 0xff] | ((uint32_t)g_sbox[(w >> 8) & 0xff] << 8) |
           ((uint32_t)g_sbox[(w >> 16) & 0xff] << 16) | ((uint32_t)g_sbox[w >> 24] << 24);
}

} /* namespace */

const uint32_t *aesoff_T0_table()
{
    std::call_once(g_once, build_tables);
    return g_T0;
}

/* Words are the little-endian load of the FIPS-197 byte string, i.e. byte 0 of w[i] (row 0 of the
 * column) is the LOW byte: RotWord is a right rotation by 8 and Rcon lands in the low byte.     */
int aesoff_key_expand(const uint8_t *key, int keybits, uint32_t rk[60])
{
    std::call_once(g_once, build_tables);
    const int nk = keybits / 32;
    if (nk != 4 && nk != 6 && nk != 8) return -1;
    const int nr = nk + 6;
    const int nwords = 4 * (nr + 1);
    for (int i = 0; i < nk; ++i)
        rk[i] = (uint32_t)key[4 * i] | ((uint32_t)key[4 * i + 1] << 8) | ((uint32_t)key[4 * i + 2] << 16) |
                ((uint32_t)key[4 * i + 3] << 24);
    uint8_t rcon = 1;
    for (int i = nk; i < nwords; ++i) {
        uint32_t t = rk[i - 1];
        if (i % nk == 0) {
            t = sub_word((t >> 8) | (t << 24)) ^ rcon;
            rcon = mul2(rcon);
        } else if (nk > 6 && i % nk == 4) {
            t = sub_word(t);
        }
        rk[i] = rk[i - nk] ^ t;
    }
    for (int i = nwords; i < 60; ++i) rk[i] = 0;
    return nr;
}

/*
 * aesni_round.c -- test helper (pin P9).
 * Exposes the host CPU's AES-NI single-round instructions so that the oracle's
 * round functions can be checked against hardware that implements FIPS-197
 * sec. 5.1 independently of any software.  Built by tests/ with `gcc -maes`;
 * the tests skip when the CPU has no `aes` flag.
 *   AESENC     : state' = MixColumns(ShiftRows(SubBytes(state))) xor rk
 *   AESENCLAST : state' =            ShiftRows(SubBytes(state))  xor rk
 *   AESKEYGENASSIST is not used: the key schedule is pinned elsewhere.
 */
#include <stdint.h>
#include <wmmintrin.h>
#include <emmintrin.h>

void aesni_enc_round(const uint8_t state[16], const uint8_t rk[16], uint8_t out[16])
{
    __m128i s = _mm_loadu_si128((const __m128i *)state);
    __m128i k = _mm_loadu_si128((const __m128i *)rk);
    _mm_storeu_si128((__m128i *)out, _mm_aesenc_si128(s, k));
}

void aesni_enc_last_round(const uint8_t state[16], const uint8_t rk[16], uint8_t out[16])
{
    __m128i s = _mm_loadu_si128((const __m128i *)state);
    __m128i k = _mm_loadu_si128((const __m128i *)rk);
    _mm_storeu_si128((__m128i *)out, _mm_aesenclast_si128(s, k));
}

/* Full cipher from caller-supplied round keys, one AES-NI instruction per round. */
void aesni_encrypt_block(const uint8_t *rk, int nr, const uint8_t in[16], uint8_t out[16])
{
    __m128i s = _mm_loadu_si128((const __m128i *)in);
    int r;
    s = _mm_xor_si128(s, _mm_loadu_si128((const __m128i *)rk));
    for (r = 1; r < nr; r++)
        s = _mm_aesenc_si128(s, _mm_loadu_si128((const __m128i *)(rk + 16 * r)));
    s = _mm_aesenclast_si128(s, _mm_loadu_si128((const __m128i *)(rk + 16 * nr)));
    _mm_storeu_si128((__m128i *)out, s);
}

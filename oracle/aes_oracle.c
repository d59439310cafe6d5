/*
 * aes_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see aes_oracle.h).
 *
 * A plain, slow, obviously-correct CPU restatement of the offload the paper's
 * servers reroute: "The GPU path performs AES" (section 6
 * Experimental setup), fixed by BASELINE.json as AES in CTR mode.  Written
 * from FIPS-197 and SP 800-38A, in their order and notation, one byte at a
 * time.  No T-tables, no intrinsics, no blocking, no typed-in S-box: every
 * constant is computed from its definition so that a reader can check each
 * function against the cited section by eye.
 */
#include "aes_oracle.h"

#include <string.h>

/* ------------------------------------------------------------------------ */
/* FIPS-197 sec. 4.2: multiplication in GF(2^8) modulo m(x) = x^8+x^4+x^3+x+1 */
/* ------------------------------------------------------------------------ */

/* sec. 4.2.1: xtime() = multiplication by x, i.e. by {02}: shift left, and if
 * the result has degree 8 reduce by subtracting (xor) m(x) = {01}{1b}.       */
uint8_t oracle_xtime(uint8_t a)
{
    uint8_t shifted = (uint8_t)(a << 1);
    if (a & 0x80)
        shifted ^= 0x1b;
    return shifted;
}

/* sec. 4.2.1: a*b by adding the xtime-multiples of a selected by the bits of b. */
uint8_t oracle_gf_mul(uint8_t a, uint8_t b)
{
    uint8_t product = 0;
    uint8_t power = a;          /* a * x^i */
    int i;
    for (i = 0; i < 8; i++) {
        if (b & (1u << i))
            product ^= power;
        power = oracle_xtime(power);
    }
    return product;
}

/* sec. 4.2 / 5.1.1: multiplicative inverse; {00} is mapped to itself.
 * Found by trying all 255 candidates -- slow on purpose.                    */
uint8_t oracle_gf_inv(uint8_t a)
{
    int b;
    if (a == 0)
        return 0;
    for (b = 1; b < 256; b++)
        if (oracle_gf_mul(a, (uint8_t)b) == 1)
            return (uint8_t)b;
    return 0; /* unreachable: GF(2^8) is a field */
}

static uint8_t rotl8(uint8_t b, int n)
{
    return (uint8_t)((b << n) | (b >> (8 - n)));
}

/* sec. 5.1.1 eq. (5.1): b'_i = b_i ^ b_(i+4) ^ b_(i+5) ^ b_(i+6) ^ b_(i+7) ^ c_i,
 * c = {63}; with indices mod 8 that is b ^ rotl(b,1..4) ^ 0x63 on the inverse. */
uint8_t oracle_sbox(uint8_t a)
{
    uint8_t b = oracle_gf_inv(a);
    return (uint8_t)(b ^ rotl8(b, 1) ^ rotl8(b, 2) ^ rotl8(b, 3) ^ rotl8(b, 4) ^ 0x63);
}

/* sec. 5.3.2: the inverse of the S-box, found by search over its 256 inputs. */
uint8_t oracle_inv_sbox(uint8_t a)
{
    int x;
    for (x = 0; x < 256; x++)
        if (oracle_sbox((uint8_t)x) == a)
            return (uint8_t)x;
    return 0; /* unreachable: the S-box is a bijection */
}

/* sec. 5.2: Rcon[j] = [x^(j-1), 00, 00, 00], powers of x = {02} in GF(2^8).  */
uint8_t oracle_rcon(int j)
{
    uint8_t r = 0x01;
    int i;
    for (i = 1; i < j; i++)
        r = oracle_xtime(r);
    return r;
}

/* The two byte substitutions are evaluated 16 times per round; cache the 256
 * values of each (still computed from the definitions above, never typed in). */
static uint8_t SBOX[256], INV_SBOX[256];
static int tables_ready = 0;

static void ensure_tables(void)
{
    int x;
    if (tables_ready)
        return;
    for (x = 0; x < 256; x++)
        SBOX[x] = oracle_sbox((uint8_t)x);
    for (x = 0; x < 256; x++)
        INV_SBOX[SBOX[x]] = (uint8_t)x;
    __atomic_store_n(&tables_ready, 1, __ATOMIC_RELEASE);
}

/* ------------------------------------------------------------------------ */
/* FIPS-197 sec. 5.1: the four transformations.  state[r + 4c] = s[r][c].     */
/* ------------------------------------------------------------------------ */

/* sec. 5.1.1 SubBytes(): S-box on each byte of the state independently.     */
void oracle_sub_bytes(uint8_t state[16])
{
    int i;
    ensure_tables();
    for (i = 0; i < 16; i++)
        state[i] = SBOX[state[i]];
}

/* sec. 5.1.2 ShiftRows(): s'[r][c] = s[r][(c + shift(r,4)) mod 4], shift(r,4)=r. */
void oracle_shift_rows(uint8_t state[16])
{
    uint8_t t[16];
    int r, c;
    for (r = 0; r < 4; r++)
        for (c = 0; c < 4; c++)
            t[r + 4 * c] = state[r + 4 * ((c + r) % 4)];
    memcpy(state, t, 16);
}

/* sec. 5.1.3 MixColumns(), eq. (5.6): each column times a(x) = {03}x^3+{01}x^2+{01}x+{02}:
 *   s'0 = 2 s0 ^ 3 s1 ^   s2 ^   s3
 *   s'1 =   s0 ^ 2 s1 ^ 3 s2 ^   s3
 *   s'2 =   s0 ^   s1 ^ 2 s2 ^ 3 s3
 *   s'3 = 3 s0 ^   s1 ^   s2 ^ 2 s3                                          */
void oracle_mix_columns(uint8_t state[16])
{
    int c;
    for (c = 0; c < 4; c++) {
        uint8_t s0 = state[0 + 4 * c], s1 = state[1 + 4 * c];
        uint8_t s2 = state[2 + 4 * c], s3 = state[3 + 4 * c];
        /* sec. 4.2.1: {02}*s = xtime(s); {03}*s = xtime(s) ^ s               */
        uint8_t d0 = oracle_xtime(s0), d1 = oracle_xtime(s1);
        uint8_t d2 = oracle_xtime(s2), d3 = oracle_xtime(s3);
        state[0 + 4 * c] = (uint8_t)(d0 ^ (d1 ^ s1) ^ s2 ^ s3);
        state[1 + 4 * c] = (uint8_t)(s0 ^ d1 ^ (d2 ^ s2) ^ s3);
        state[2 + 4 * c] = (uint8_t)(s0 ^ s1 ^ d2 ^ (d3 ^ s3));
        state[3 + 4 * c] = (uint8_t)((d0 ^ s0) ^ s1 ^ s2 ^ d3);
    }
}

/* sec. 5.1.4 AddRoundKey(): column c of the state xor word c of the round key. */
void oracle_add_round_key(uint8_t state[16], const uint8_t rk16[16])
{
    int i;
    for (i = 0; i < 16; i++)
        state[i] ^= rk16[i];
}

/* sec. 5.3.2 InvSubBytes().                                                  */
void oracle_inv_sub_bytes(uint8_t state[16])
{
    int i;
    ensure_tables();
    for (i = 0; i < 16; i++)
        state[i] = INV_SBOX[state[i]];
}

/* sec. 5.3.1 InvShiftRows(): s'[r][(c + r) mod 4] = s[r][c].                 */
void oracle_inv_shift_rows(uint8_t state[16])
{
    uint8_t t[16];
    int r, c;
    for (r = 0; r < 4; r++)
        for (c = 0; c < 4; c++)
            t[r + 4 * ((c + r) % 4)] = state[r + 4 * c];
    memcpy(state, t, 16);
}

/* sec. 5.3.3 InvMixColumns(), eq. (5.10): a^-1(x) = {0b}x^3+{0d}x^2+{09}x+{0e}. */
void oracle_inv_mix_columns(uint8_t state[16])
{
    int c;
    for (c = 0; c < 4; c++) {
        uint8_t s0 = state[0 + 4 * c], s1 = state[1 + 4 * c];
        uint8_t s2 = state[2 + 4 * c], s3 = state[3 + 4 * c];
        state[0 + 4 * c] = (uint8_t)(oracle_gf_mul(0x0e, s0) ^ oracle_gf_mul(0x0b, s1) ^
                                     oracle_gf_mul(0x0d, s2) ^ oracle_gf_mul(0x09, s3));
        state[1 + 4 * c] = (uint8_t)(oracle_gf_mul(0x09, s0) ^ oracle_gf_mul(0x0e, s1) ^
                                     oracle_gf_mul(0x0b, s2) ^ oracle_gf_mul(0x0d, s3));
        state[2 + 4 * c] = (uint8_t)(oracle_gf_mul(0x0d, s0) ^ oracle_gf_mul(0x09, s1) ^
                                     oracle_gf_mul(0x0e, s2) ^ oracle_gf_mul(0x0b, s3));
        state[3 + 4 * c] = (uint8_t)(oracle_gf_mul(0x0b, s0) ^ oracle_gf_mul(0x0d, s1) ^
                                     oracle_gf_mul(0x09, s2) ^ oracle_gf_mul(0x0e, s3));
    }
}

/* ------------------------------------------------------------------------ */
/* FIPS-197 sec. 5.2 KeyExpansion() (Figure 11), on words of four bytes.      */
/* ------------------------------------------------------------------------ */
int oracle_key_expand(const uint8_t *key, int keybits, uint8_t *rk)
{
    int Nk, Nr, i, b;
    uint8_t *w = rk;            /* w[i] is the four bytes rk[4i .. 4i+3]      */

    if (keybits == 128)      { Nk = 4; Nr = 10; }
    else if (keybits == 192) { Nk = 6; Nr = 12; }
    else if (keybits == 256) { Nk = 8; Nr = 14; }
    else return -1;
    ensure_tables();

    /* while (i < Nk) w[i] = word(key[4i], key[4i+1], key[4i+2], key[4i+3])   */
    for (i = 0; i < Nk; i++)
        for (b = 0; b < 4; b++)
            w[4 * i + b] = key[4 * i + b];

    /* while (i < Nb*(Nr+1)) ...                                              */
    for (i = Nk; i < 4 * (Nr + 1); i++) {
        uint8_t temp[4];
        for (b = 0; b < 4; b++)
            temp[b] = w[4 * (i - 1) + b];
        if (i % Nk == 0) {
            /* temp = SubWord(RotWord(temp)) xor Rcon[i/Nk]
             * RotWord([a0,a1,a2,a3]) = [a1,a2,a3,a0]                         */
            uint8_t a0 = temp[0];
            temp[0] = temp[1]; temp[1] = temp[2]; temp[2] = temp[3]; temp[3] = a0;
            for (b = 0; b < 4; b++)
                temp[b] = SBOX[temp[b]];
            temp[0] ^= oracle_rcon(i / Nk);
        } else if (Nk > 6 && i % Nk == 4) {
            /* temp = SubWord(temp)                                           */
            for (b = 0; b < 4; b++)
                temp[b] = SBOX[temp[b]];
        }
        /* w[i] = w[i-Nk] xor temp                                            */
        for (b = 0; b < 4; b++)
            w[4 * i + b] = (uint8_t)(w[4 * (i - Nk) + b] ^ temp[b]);
    }
    return Nr;
}

/* ------------------------------------------------------------------------ */
/* FIPS-197 sec. 5.1 Cipher() (Figure 5) and sec. 5.3 InvCipher() (Figure 12). */
/* ------------------------------------------------------------------------ */
void oracle_encrypt_block(const uint8_t *rk, int nr, const uint8_t in[16], uint8_t out[16])
{
    uint8_t state[16];
    int round;
    memcpy(state, in, 16);                       /* state = in                */
    oracle_add_round_key(state, rk);             /* AddRoundKey(w[0, Nb-1])   */
    for (round = 1; round <= nr - 1; round++) {
        oracle_sub_bytes(state);
        oracle_shift_rows(state);
        oracle_mix_columns(state);
        oracle_add_round_key(state, rk + 16 * round);
    }
    oracle_sub_bytes(state);
    oracle_shift_rows(state);
    oracle_add_round_key(state, rk + 16 * nr);
    memcpy(out, state, 16);                      /* out = state               */
}

void oracle_decrypt_block(const uint8_t *rk, int nr, const uint8_t in[16], uint8_t out[16])
{
    uint8_t state[16];
    int round;
    memcpy(state, in, 16);
    oracle_add_round_key(state, rk + 16 * nr);
    for (round = nr - 1; round >= 1; round--) {
        oracle_inv_shift_rows(state);
        oracle_inv_sub_bytes(state);
        oracle_add_round_key(state, rk + 16 * round);
        oracle_inv_mix_columns(state);
    }
    oracle_inv_shift_rows(state);
    oracle_inv_sub_bytes(state);
    oracle_add_round_key(state, rk);
    memcpy(out, state, 16);
}

/* ------------------------------------------------------------------------ */
/* SP 800-38A sec. 6.5 CTR mode, appendix B.1 standard incrementing function  */
/* with m = 128: the whole block is one big-endian integer, wrapping mod 2^128 */
/* (reading R4; OpenSSL and `cryptography` do the same).            */
/* ------------------------------------------------------------------------ */

/* out = (icb + add) mod 2^128: schoolbook addition from the last byte up.    */
void oracle_ctr_add(const uint8_t icb[16], uint64_t add, uint8_t out[16])
{
    unsigned carry = 0;
    int i;
    for (i = 15; i >= 0; i--) {
        unsigned addend = (unsigned)(add & 0xff);
        unsigned sum = (unsigned)icb[i] + addend + carry;
        out[i] = (uint8_t)(sum & 0xff);
        carry = sum >> 8;
        add >>= 8;
    }
}

/* T <- (T + 1) mod 2^128.                                                    */
static void ctr_increment(uint8_t T[16])
{
    int i;
    for (i = 15; i >= 0; i--) {
        T[i] = (uint8_t)(T[i] + 1);
        if (T[i] != 0)
            break;              /* no carry into the next byte               */
    }
}

void oracle_ctr_at(const uint8_t *rk, int nr, const uint8_t icb[16], uint64_t block_offset,
                   const uint8_t *src, uint8_t *dst, size_t len)
{
    uint8_t T[16], O[16];
    size_t done = 0;
    oracle_ctr_add(icb, block_offset, T);        /* T_1 of this window        */
    while (done < len) {
        size_t u = len - done < 16 ? len - done : 16;
        size_t i;
        oracle_encrypt_block(rk, nr, T, O);      /* O_j = CIPH_K(T_j)         */
        for (i = 0; i < u; i++)                  /* C_j = P_j xor MSB_u(O_j)  */
            dst[done + i] = (uint8_t)(src[done + i] ^ O[i]);
        ctr_increment(T);                        /* T_{j+1}                   */
        done += u;
    }
}

void oracle_ctr(const uint8_t *rk, int nr, const uint8_t icb[16],
                const uint8_t *src, uint8_t *dst, size_t len)
{
    oracle_ctr_at(rk, nr, icb, 0, src, dst, len);
}

/* ------------------------------------------------------------------------ */
/* SP 800-38A sec. 6.1 ECB mode and sec. 6.2 CBC mode, whole blocks only (the   */
/* standard defines both on a sequence of complete blocks; padding is the       */
/* caller's business, sec. 5.2 / appendix A).  DESIGN.md reading R13: the paper */
/* "performs AES" without naming a mode; CTR is the mode the     */
/* benchmark fixes, ECB and CBC decryption are the other two modes in which     */
/* every block can be computed independently.         */
/* ------------------------------------------------------------------------ */

/* ECB encryption: C_j = CIPH_K(P_j), j = 1..n (sec. 6.1).                    */
void oracle_ecb_encrypt(const uint8_t *rk, int nr, const uint8_t *src, uint8_t *dst, size_t nblocks)
{
    size_t j;
    for (j = 0; j < nblocks; j++) {
        uint8_t P[16], C[16];
        memcpy(P, src + 16 * j, 16);
        oracle_encrypt_block(rk, nr, P, C);
        memcpy(dst + 16 * j, C, 16);
    }
}

/* ECB decryption: P_j = CIPH^-1_K(C_j), j = 1..n (sec. 6.1).                 */
void oracle_ecb_decrypt(const uint8_t *rk, int nr, const uint8_t *src, uint8_t *dst, size_t nblocks)
{
    size_t j;
    for (j = 0; j < nblocks; j++) {
        uint8_t C[16], P[16];
        memcpy(C, src + 16 * j, 16);
        oracle_decrypt_block(rk, nr, C, P);
        memcpy(dst + 16 * j, P, 16);
    }
}

/* CBC encryption: C_1 = CIPH_K(P_1 xor IV); C_j = CIPH_K(P_j xor C_{j-1}), j = 2..n
 * (sec. 6.2).  Sequential by definition; here so that tests have ciphertexts to
 * decrypt and a round trip to check -- the GPU path only decrypts.            */
void oracle_cbc_encrypt(const uint8_t *rk, int nr, const uint8_t iv[16], const uint8_t *src, uint8_t *dst,
                        size_t nblocks)
{
    uint8_t prev[16];
    size_t j;
    int i;
    memcpy(prev, iv, 16);                        /* "C_0" = IV                 */
    for (j = 0; j < nblocks; j++) {
        uint8_t X[16], C[16];
        for (i = 0; i < 16; i++)
            X[i] = (uint8_t)(src[16 * j + i] ^ prev[i]);
        oracle_encrypt_block(rk, nr, X, C);
        memcpy(dst + 16 * j, C, 16);
        memcpy(prev, C, 16);
    }
}

/* CBC decryption: P_1 = CIPH^-1_K(C_1) xor IV; P_j = CIPH^-1_K(C_j) xor C_{j-1},
 * j = 2..n (sec. 6.2).  dst may equal src (the previous ciphertext block is
 * kept in a local copy).                                                       */
void oracle_cbc_decrypt(const uint8_t *rk, int nr, const uint8_t iv[16], const uint8_t *src, uint8_t *dst,
                        size_t nblocks)
{
    uint8_t prev[16];
    size_t j;
    int i;
    memcpy(prev, iv, 16);
    for (j = 0; j < nblocks; j++) {
        uint8_t C[16], X[16];
        memcpy(C, src + 16 * j, 16);
        oracle_decrypt_block(rk, nr, C, X);
        for (i = 0; i < 16; i++)
            dst[16 * j + i] = (uint8_t)(X[i] ^ prev[i]);
        memcpy(prev, C, 16);
    }
}

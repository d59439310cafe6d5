/*
 * aes_oracle.h -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, byte-level reference for what the GPU hot path computes:
 * FIPS-197 AES (Nk = 4/6/8) and SP 800-38A section 6.5 CTR mode on top of it.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code, table, header or
 * constant generator with paper_2607_02630_b200/csrc (the CUDA path).
 *
 * What it follows (the reading of PAPER.md:224
 * "The GPU path performs AES [OpenSSL Project, 2026]" that BASELINE.json fixes
 * as AES-128/256 in CTR mode):
 *   - GF(2^8) arithmetic modulo x^8+x^4+x^3+x+1            FIPS-197 sec. 4
 *   - S-box computed as affine(inverse(a))                 FIPS-197 sec. 5.1.1
 *   - KeyExpansion                                         FIPS-197 sec. 5.2
 *   - Cipher / InvCipher                                   FIPS-197 sec. 5.1 / 5.3
 *   - CTR with a 128-bit big-endian incrementing function  SP 800-38A sec. 6.5, B.1
 *   - ECB and CBC on whole blocks          SP 800-38A sec. 6.1, 6.2
 *
 * Pins: every function below is pinned by tests/test_oracle_*.py (-m "not gpu")
 * against the standards' printed vectors (tests/golden/), OpenSSL libcrypto,
 * Python `cryptography`, host AES-NI single rounds, closed forms and
 * invariants.  No function here is "parity unpinned".
 */
#ifndef AES_ORACLE_H
#define AES_ORACLE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- GF(2^8) and the S-box (FIPS-197 sec. 4.2, 5.1.1) ------------------- */
uint8_t oracle_xtime(uint8_t a);               /* a * {02}                    */
uint8_t oracle_gf_mul(uint8_t a, uint8_t b);   /* a * b in GF(2^8)            */
uint8_t oracle_gf_inv(uint8_t a);              /* a^-1, with inv(0) = 0       */
uint8_t oracle_sbox(uint8_t a);                /* SubBytes on one byte        */
uint8_t oracle_inv_sbox(uint8_t a);            /* InvSubBytes on one byte     */
uint8_t oracle_rcon(int j);                    /* {02}^(j-1), j >= 1          */

/* ---- round transformations on a 16-byte state (FIPS-197 sec. 5.1) -------
 * The state is passed in the input/output byte order of the standard:
 * s[r][c] = state[r + 4c] (sec. 3.4).                                        */
void oracle_sub_bytes(uint8_t state[16]);
void oracle_shift_rows(uint8_t state[16]);
void oracle_mix_columns(uint8_t state[16]);
void oracle_add_round_key(uint8_t state[16], const uint8_t rk16[16]);
void oracle_inv_sub_bytes(uint8_t state[16]);
void oracle_inv_shift_rows(uint8_t state[16]);
void oracle_inv_mix_columns(uint8_t state[16]);

/* ---- key schedule (FIPS-197 sec. 5.2) ------------------------------------
 * keybits in {128,192,256}.  Writes 16*(Nr+1) bytes to rk: round key r is
 * rk[16r .. 16r+15], its word c is bytes 4c..4c+3 (column c of the state).
 * Returns Nr (10/12/14), or -1 if keybits is not one of the three.          */
int oracle_key_expand(const uint8_t *key, int keybits, uint8_t *rk);

/* ---- block cipher (FIPS-197 sec. 5.1, 5.3) ------------------------------- */
void oracle_encrypt_block(const uint8_t *rk, int nr, const uint8_t in[16], uint8_t out[16]);
void oracle_decrypt_block(const uint8_t *rk, int nr, const uint8_t in[16], uint8_t out[16]);

/* ---- CTR (SP 800-38A sec. 6.5) -------------------------------------------
 * T_1 = icb, T_{j+1} = (T_j + 1) mod 2^128 as a big-endian integer
 * (the standard incrementing function of appendix B.1 with m = 128);
 * O_j = Cipher_K(T_j); C_j = P_j xor O_j; a final partial block of u bytes
 * uses the u most significant (first) bytes of O_n.  dst may equal src.
 * oracle_ctr_at starts the counter at icb + block_offset, i.e. it computes
 * bytes [16*block_offset, 16*block_offset + len) of the stream.             */
void oracle_ctr(const uint8_t *rk, int nr, const uint8_t icb[16],
                const uint8_t *src, uint8_t *dst, size_t len);
void oracle_ctr_at(const uint8_t *rk, int nr, const uint8_t icb[16], uint64_t block_offset,
                   const uint8_t *src, uint8_t *dst, size_t len);

/* icb + add (mod 2^128, big-endian) -> out.  Exposed so tests can pin it.   */
void oracle_ctr_add(const uint8_t icb[16], uint64_t add, uint8_t out[16]);

/* ---- ECB and CBC (SP 800-38A sec. 6.1, 6.2) -------------------------------
 * Whole blocks only: nblocks x 16 bytes, no padding (the standard defines both
 * modes on complete blocks).  ECB: C_j = CIPH_K(P_j) / P_j = CIPH^-1_K(C_j).
 * CBC: C_1 = CIPH_K(P_1 xor IV), C_j = CIPH_K(P_j xor C_{j-1});
 *      P_1 = CIPH^-1_K(C_1) xor IV, P_j = CIPH^-1_K(C_j) xor C_{j-1}.
 * dst may equal src in all four.  The GPU path has ECB both ways and CBC
 * decryption (every block independent); CBC encryption is sequential by
 * definition and is here for the tests' round trips.                          */
void oracle_ecb_encrypt(const uint8_t *rk, int nr, const uint8_t *src, uint8_t *dst, size_t nblocks);
void oracle_ecb_decrypt(const uint8_t *rk, int nr, const uint8_t *src, uint8_t *dst, size_t nblocks);
void oracle_cbc_encrypt(const uint8_t *rk, int nr, const uint8_t iv[16], const uint8_t *src, uint8_t *dst,
                        size_t nblocks);
void oracle_cbc_decrypt(const uint8_t *rk, int nr, const uint8_t iv[16], const uint8_t *src, uint8_t *dst,
                        size_t nblocks);

#ifdef __cplusplus
}
#endif
#endif /* AES_ORACLE_H */

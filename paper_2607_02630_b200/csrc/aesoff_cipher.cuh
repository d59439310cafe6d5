/*
 * aesoff_cipher.cuh -- the AES-CTR arithmetic of the sm_100a path (steps a4-a6 of SURVEY.md
 * section 8(a)): shared-memory table layout, table fill, and one "row" of CTR by one warp.
 * Included by aesoff_kernels.cu (engine kernel).
 *
 *   FIPS-197 Cipher() with the SubBytes/ShiftRows/MixColumns of a round folded into four
 *   256-entry word tables (the classical "T-table" form of sec. 5.1: column j of a round's output
 *   is T0[s0,j] ^ T1[s1,j+1] ^ T2[s2,j+2] ^ T3[s3,j+3] ^ roundkey), SP 800-38A sec. 6.5 CTR around it.
 *
 * B200 specifics (DESIGN.md sections 5-7):
 *   - The binding unit is the shared-memory crossbar: 32 four-byte lookups per clock per SM.  Each of
 *     the four tables is therefore replicated once per bank (lane l only ever reads bank l), which
 *     makes every LDS conflict-free by construction: 4 x 256 x 32 x 4 B = 128 KiB per SM.
 *   - Entries sit at a 256-byte stride (two tables interleaved per 64 KiB region) so that one PRMT
 *     builds the whole lookup address  (byte_k(x) << 8) | lane*4 | region_base.
 *   - CTR structure: a warp works on one "row" = the 256 counter values that share the upper 120
 *     counter bits.  Everything of rounds 1 and 2 that depends only on those bits is computed once
 *     per row; per block round 1 is ONE lookup and round 2 FOUR: 133 lookups per AES-128 block in
 *     the row's step instead of 160, 197 instead of 224 for AES-256 -- 135.3 / 199.3 once the row
 *     set-up (27 + 10 lookups per lane for a pair of rows = 16 blocks) is counted in, the figure
 *     bench.py's roofline uses.
 *   - Payload is read/written with 128-bit L2-only accesses (ld.global.cg / st.global.cg): a
 *     persistent kernel never gets its L1 invalidated, so a recycled request buffer must not hit L1.
 */
#ifndef AESOFF_CIPHER_CUH
#define AESOFF_CIPHER_CUH

#include <cuda_runtime.h>
#include <stdint.h>

#include "aesoff_shared.h"

namespace aesoff {

/* ------------------------------------------------------------------------------------------ */
/* shared-memory table layout                                                                  */
/* ------------------------------------------------------------------------------------------ */
constexpr int OFF_T0 = 0;
constexpr int OFF_T1 = 128;
constexpr int OFF_T2 = 65536;
constexpr int OFF_T3 = 65536 + 128;
constexpr uint32_t TABLE_BYTES = 131072;
/* The decryption modes (ECB, CBC) run the equivalent inverse cipher (FIPS-197 sec. 5.3.5)
 * out of ONE more table, Td0, again one replica per bank: entry x of lane l at TD_OFF + x * 128 + l * 4, 32 KiB
 * behind the four encryption tables (all the shared memory an SM has left).  Td1..Td3 are byte rotations done in
 * registers and the address needs a shift and a mask: these modes are bound by the ALU pipe, not by lookups.    */
constexpr uint32_t TD_OFF = TABLE_BYTES;
constexpr uint32_t TD_BYTES = 32768;

template <int OFF>
__device__ __forceinline__ uint32_t lds_off(uint32_t a)
{
    uint32_t v;
    asm("ld.shared.u32 %0, [%1+%2];" : "=r"(v) : "r"(a), "n"(OFF));
    return v;
}
__device__ __forceinline__ void sts(uint32_t a, uint32_t v)
{
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
/* (byte K of x) << 8 | ybase, where ybase = region_base | lane*4 and region_base % 65536 == 0 */
template <int K>
__device__ __forceinline__ uint32_t taddr(uint32_t x, uint32_t ybase)
{
    return __byte_perm(x, ybase, 0x7604 | (K << 4));
}
#define TL(T, K, x) lds_off<OFF_T##T>(taddr<K>((x), ybase))

__device__ __forceinline__ uint32_t bswap32(uint32_t x) { return __byte_perm(x, 0, 0x0123); }
__device__ __forceinline__ uint32_t rotl32(uint32_t x, int n) { return __funnelshift_l(x, x, n); }
__device__ __forceinline__ uint32_t bitsel(uint32_t a, uint32_t b, uint32_t m) { return (a & m) | (b & ~m); }

/* at most one block per request takes this path, so it is kept out of line */
static __device__ __noinline__ void store_partial(const uint8_t *src, uint8_t *dst, uint32_t o0, uint32_t o1, uint32_t o2,
                                           uint32_t o3, uint32_t u)
{
#pragma unroll 1
    for (uint32_t i = 0; i < u; ++i) {
        const uint32_t w = (i < 8) ? (i < 4 ? o0 : o1) : (i < 12 ? o2 : o3);
        const uint8_t ks = (uint8_t)(w >> (8u * (i & 3u)));
        const uint8_t pt = __ldcg(src + i);
        __stcg(dst + i, (uint8_t)(pt ^ ks));
    }
}


/* ------------------------------------------------------------------------------------------ */
/* table fill (step a0): T0 comes from global memory (256 words built by the host from the     */
/* S-box definition, aesoff_keys.cpp); T1..T3 are its byte rotations; 32 replicas each         */
/* ------------------------------------------------------------------------------------------ */
/* Called by the CTA's first `nthreads` threads (the worker warps; a multiple of 32); they meet on
 * named barrier 2, and the tables are complete when it returns.                                 */
__device__ __forceinline__ void fill_barrier(uint32_t nthreads)
{
    asm volatile("bar.sync 2, %0;" ::"r"(nthreads) : "memory");
}
__device__ __forceinline__ void fill_tables(uint32_t tbase, const uint32_t *T0, uint32_t tid, uint32_t nthreads)
{
    /* one global read per entry, staged in what becomes lane 0's replica of T0 ... */
    for (uint32_t i = tid; i < 256u; i += nthreads) sts(tbase + i * 256u + OFF_T0, __ldg(T0 + i));
    fill_barrier(nthreads);
    /* ... then replicated and rotated out of shared memory */
    for (uint32_t idx = tid; idx < 256u * 32u; idx += nthreads) {
        const uint32_t i = idx >> 5, l = idx & 31u;
        uint32_t t0;
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(t0) : "r"(tbase + i * 256u) : "memory");
        const uint32_t a = tbase + i * 256u + l * 4u;
        if (l != 0u) sts(a + OFF_T0, t0);
        sts(a + OFF_T1, rotl32(t0, 8));
        sts(a + OFF_T2, rotl32(t0, 16));
        sts(a + OFF_T3, rotl32(t0, 24));
    }
    fill_barrier(nthreads);
}

/* Td0 replicas (global table at Td0[0..255]); called like fill_tables, after it */
__device__ __forceinline__ void fill_td(uint32_t tbase, const uint32_t *Td0, uint32_t tid, uint32_t nthreads)
{
    for (uint32_t idx = tid; idx < 256u * 32u; idx += nthreads) sts(tbase + TD_OFF + idx * 4u, __ldg(Td0 + (idx >> 5)));
    fill_barrier(nthreads);
}
/* Td0[byte K of x] out of this lane's replica; ybd = (tbase + TD_OFF) | lane * 4 */
template <int K>
__device__ __forceinline__ uint32_t td(uint32_t x, uint32_t ybd)
{
    /* The inverse rounds are bound by the ALU pipe (ncu, profiles/r3_ncu_modes.md: 97.7 % busy with shift + mask-or per
     * address), so the address costs that pipe ONE instruction -- PRMT pulls the byte out -- and the scaling by the
     * 128-byte entry stride plus the base goes to the FMA pipe as an integer multiply-add, which otherwise idles.     */
    const uint32_t b = __byte_perm(x, 0u, 0x4440u | K);
    uint32_t a, v;
    asm("mad.lo.u32 %0, %1, 128, %2;" : "=r"(a) : "r"(b), "r"(ybd));
    asm("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint32_t xor_bytes(uint32_t t) /* InvSubBytes(x) from Td0[x] */
{
    t ^= t >> 16;
    return (t ^ (t >> 8)) & 0xffu;
}
/* one column of an inverse round: InvShiftRows moves row r right by r columns */
__device__ __forceinline__ uint32_t td_col(uint32_t a, uint32_t b, uint32_t c, uint32_t d, uint32_t ybd)
{
    return td<0>(a, ybd) ^ rotl32(td<1>(b, ybd), 8) ^ rotl32(td<2>(c, ybd), 16) ^ rotl32(td<3>(d, ybd), 24);
}
__device__ __forceinline__ uint32_t tdlast_col(uint32_t a, uint32_t b, uint32_t c, uint32_t d, uint32_t ybd)
{
    return xor_bytes(td<0>(a, ybd)) | (xor_bytes(td<1>(b, ybd)) << 8) | (xor_bytes(td<2>(c, ybd)) << 16) |
           (xor_bytes(td<3>(d, ybd)) << 24);
}
/* Round keys of the equivalent inverse cipher (sec. 5.3.5): dw[r] = InvMixColumns(w[r]) for 0 < r < Nr, word by word:
 * InvMixColumns of a column is Td0[S[a0]] ^ rot(Td0[S[a1]]) ^ ..., S[a] being byte 1 of T0[a].                  */
__device__ __forceinline__ uint32_t inv_mix_word(uint32_t w, uint32_t ybase, uint32_t ybd)
{
    const uint32_t s0 = TL(0, 0, w) >> 8, s1 = TL(0, 1, w) >> 8, s2 = TL(0, 2, w) >> 8, s3 = TL(0, 3, w) >> 8;
    return td<0>(s0, ybd) ^ rotl32(td<0>(s1, ybd), 8) ^ rotl32(td<0>(s2, ybd), 16) ^ rotl32(td<0>(s3, ybd), 24);
}

/* ------------------------------------------------------------------------------------------ */
/* key expansion (step a1) for keys that arrive raw in a descriptor: FIPS-197 sec. 5.2          */
/* ------------------------------------------------------------------------------------------ */
/* SubWord out of this lane's replica of T0: S[x] is byte 1 (and 2) of T0[x].                   */
__device__ __forceinline__ uint32_t sub_word(uint32_t w, uint32_t ybase)
{
    const uint32_t t0 = TL(0, 0, w), t1 = TL(0, 1, w), t2 = TL(0, 2, w), t3 = TL(0, 3, w);
    return ((t0 >> 8) & 0xffu) | (t1 & 0xff00u) | (t2 & 0xff0000u) | ((t3 << 16) & 0xff000000u);
}
/* key: Nk little-endian-loaded words of the cipher key; out: 4 (Nk + 7) words in global memory.
 * Words are little-endian loads of the FIPS-197 byte string, so RotWord is a right rotation by 8
 * and Rcon lands in the low byte.  One thread, one serial chain of 10 (Nk = 4), 8 (Nk = 6) or 13
 * (Nk = 8) SubWords: well under a microsecond, against a PCIe round trip for shipping 240 bytes. */
template <int NK>
__device__ __forceinline__ void key_expand(uint32_t ybase, const uint32_t *key, uint32_t *out)
{
    uint32_t w[NK];
#pragma unroll
    for (int i = 0; i < NK; ++i) {
        w[i] = key[i];
        __stcg(out + i, w[i]);
    }
    uint32_t rcon = 1;
#pragma unroll
    for (int i = NK; i < 4 * (NK + 7); ++i) {
        uint32_t t = w[(i - 1) % NK];
        if (i % NK == 0) {
            t = sub_word(__funnelshift_r(t, t, 8), ybase) ^ rcon;
            rcon = ((rcon << 1) ^ ((rcon & 0x80u) ? 0x11bu : 0u)) & 0xffu; /* xtime, sec. 4.2.1 */
        } else if (NK > 6 && i % NK == 4) {
            t = sub_word(t, ybase);
        }
        w[i % NK] ^= t;
        __stcg(out + i, w[i % NK]);
    }
}

/* ------------------------------------------------------------------------------------------ */
/* one row: the (up to) 256 blocks whose counter blocks share bytes 0..14                      */
/* ------------------------------------------------------------------------------------------ */
/* Everything of rounds 0..2 that the 256 blocks of a row have in common (27 lookups).          */
struct RowConst {
    uint32_t K1_0;                   /* round-1 column 0 without the T3[byte 15] term          */
    uint32_t K2_0, K2_1, K2_2, K2_3; /* round-2 columns without the terms fed by column 0      */
    uint32_t a3;                     /* address of T3[state byte 15] for last counter byte = lane */
    uint32_t C1, s3;                 /* round-1 column 1 and round-0 word 3: all that counter byte 14 reaches */
};

/* U0..U3: the counter block with its last byte zero, as four little-endian-loaded words;
 * rk4: round keys in shared memory (uint4 per round).                                          */
__device__ __forceinline__ RowConst row_setup(uint32_t ybase, const uint4 *rk4, uint32_t U0, uint32_t U1, uint32_t U2,
                                              uint32_t U3, uint32_t lane)
{
    const uint4 k0 = rk4[0], k1 = rk4[1], k2 = rk4[2];
    /* round 0 (AddRoundKey) on the row's common counter block */
    const uint32_t s0 = U0 ^ k0.x, s1 = U1 ^ k0.y, s2 = U2 ^ k0.z, s3 = U3 ^ k0.w;
    RowConst rc;
    /* round 1: columns 1..3 do not see the last counter byte at all, column 0 sees it through T3 */
    rc.K1_0 = TL(0, 0, s0) ^ TL(1, 1, s1) ^ TL(2, 2, s2) ^ k1.x;
    const uint32_t C1 = TL(0, 0, s1) ^ TL(1, 1, s2) ^ TL(2, 2, s3) ^ TL(3, 3, s0) ^ k1.y;
    const uint32_t C2 = TL(0, 0, s2) ^ TL(1, 1, s3) ^ TL(2, 2, s0) ^ TL(3, 3, s1) ^ k1.z;
    const uint32_t C3 = TL(0, 0, s3) ^ TL(1, 1, s0) ^ TL(2, 2, s1) ^ TL(3, 3, s2) ^ k1.w;
    /* round 2: per column, the three lookups fed by the constant columns C1..C3 */
    rc.K2_0 = TL(1, 1, C1) ^ TL(2, 2, C2) ^ TL(3, 3, C3) ^ k2.x;
    rc.K2_1 = TL(0, 0, C1) ^ TL(1, 1, C2) ^ TL(2, 2, C3) ^ k2.y;
    rc.K2_2 = TL(0, 0, C2) ^ TL(1, 1, C3) ^ TL(3, 3, C1) ^ k2.z;
    rc.K2_3 = TL(0, 0, C3) ^ TL(2, 2, C1) ^ TL(3, 3, C2) ^ k2.w;
    /* the last counter byte (lane + 32k) is xored into the table index: lane here, k per block */
    rc.a3 = taddr<3>(s3, ybase) ^ (lane << 8);
    rc.C1 = C1;
    rc.s3 = s3;
    return rc;
}

/* The next row of the same request when only counter byte 14 changed (no carry out of it): that byte
 * enters round 1 through ONE lookup of column 1, and column 1 enters round 2 through one lookup per
 * column -- 10 lookups (old and new term each) instead of the 27 of a full set-up.
 * U3_new: word 3 of the new row's counter block (last byte zero), little-endian loaded.            */
__device__ __forceinline__ void row_step(RowConst &rc, uint32_t ybase, uint32_t k0w, uint32_t U3_new)
{
    const uint32_t s3n = U3_new ^ k0w;
    const uint32_t C1n = rc.C1 ^ TL(2, 2, rc.s3) ^ TL(2, 2, s3n);
    rc.K2_0 ^= TL(1, 1, rc.C1) ^ TL(1, 1, C1n);
    rc.K2_1 ^= TL(0, 0, rc.C1) ^ TL(0, 0, C1n);
    rc.K2_2 ^= TL(3, 3, rc.C1) ^ TL(3, 3, C1n);
    rc.K2_3 ^= TL(2, 2, rc.C1) ^ TL(2, 2, C1n);
    rc.C1 = C1n;
    rc.s3 = s3n; /* byte 3 of s3 (counter byte 15, zero here) is unchanged, and so is rc.a3 */
}

/* NB blocks per lane: L = lane + 32 (kb + b), b = 0..NB-1.
 * src_row  address the block with last counter byte 0 would have (may lie before the payload)
 * lo_L     first valid value of the last counter byte in this row (non-zero only in row 0)
 * row_bytes  payload bytes from src_row to the end of the payload, capped at 4096               */
template <int NB>
__device__ __forceinline__ void row_blocks(const RowConst &rc, uint32_t ybase, const uint4 *rk4, int nr,
                                           const uint8_t *src_row, uint8_t *dst_row, uint32_t lo_L,
                                           uint32_t row_bytes, uint32_t lane, uint32_t kb)
{
    uint4 p[NB];
    uint32_t st[NB][4];
    bool full[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        const uint32_t L = lane + 32u * (kb + b), off = L * 16u;
        full[b] = (L >= lo_L) && (off + 16u <= row_bytes);
        p[b] = make_uint4(0, 0, 0, 0);
        if (full[b]) p[b] = __ldcg(reinterpret_cast<const uint4 *>(src_row + off));
    }
    /* rounds 1 and 2: 1 + 4 lookups per block */
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        const uint32_t r1 = rc.K1_0 ^ lds_off<OFF_T3>(rc.a3 ^ ((kb + b) << 13));
        st[b][0] = rc.K2_0 ^ TL(0, 0, r1);
        st[b][1] = rc.K2_1 ^ TL(3, 3, r1);
        st[b][2] = rc.K2_2 ^ TL(2, 2, r1);
        st[b][3] = rc.K2_3 ^ TL(1, 1, r1);
    }
    /* rounds 3 .. Nr-1: 16 lookups per block per round */
#pragma unroll 1
    for (int r = 3; r < nr; ++r) {
        const uint4 kk = rk4[r];
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const uint32_t x0 = st[b][0], x1 = st[b][1], x2 = st[b][2], x3 = st[b][3];
            st[b][0] = TL(0, 0, x0) ^ TL(1, 1, x1) ^ TL(2, 2, x2) ^ TL(3, 3, x3) ^ kk.x;
            st[b][1] = TL(0, 0, x1) ^ TL(1, 1, x2) ^ TL(2, 2, x3) ^ TL(3, 3, x0) ^ kk.y;
            st[b][2] = TL(0, 0, x2) ^ TL(1, 1, x3) ^ TL(2, 2, x0) ^ TL(3, 3, x1) ^ kk.z;
            st[b][3] = TL(0, 0, x3) ^ TL(1, 1, x0) ^ TL(2, 2, x1) ^ TL(3, 3, x2) ^ kk.w;
        }
    }
    /* final round: SubBytes + ShiftRows + AddRoundKey.  S[x] is read out of the T entries:
     * T3 has it in byte 0, T0 in bytes 1 and 2, T1 in byte 3.                                */
    const uint4 kk = rk4[nr];
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        const uint32_t x0 = st[b][0], x1 = st[b][1], x2 = st[b][2], x3 = st[b][3];
        uint32_t o[4];
        o[0] = bitsel(bitsel(TL(3, 0, x0), TL(0, 1, x1), 0x000000ffu),
                      bitsel(TL(0, 2, x2), TL(1, 3, x3), 0x00ff0000u), 0x0000ffffu) ^ kk.x;
        o[1] = bitsel(bitsel(TL(3, 0, x1), TL(0, 1, x2), 0x000000ffu),
                      bitsel(TL(0, 2, x3), TL(1, 3, x0), 0x00ff0000u), 0x0000ffffu) ^ kk.y;
        o[2] = bitsel(bitsel(TL(3, 0, x2), TL(0, 1, x3), 0x000000ffu),
                      bitsel(TL(0, 2, x0), TL(1, 3, x1), 0x00ff0000u), 0x0000ffffu) ^ kk.z;
        o[3] = bitsel(bitsel(TL(3, 0, x3), TL(0, 1, x0), 0x000000ffu),
                      bitsel(TL(0, 2, x1), TL(1, 3, x2), 0x00ff0000u), 0x0000ffffu) ^ kk.w;
        const uint32_t L = lane + 32u * (kb + b), off = L * 16u;
        if (full[b]) {
            uint4 c;
            c.x = p[b].x ^ o[0];
            c.y = p[b].y ^ o[1];
            c.z = p[b].z ^ o[2];
            c.w = p[b].w ^ o[3];
            __stcg(reinterpret_cast<uint4 *>(dst_row + off), c);
        } else if (L >= lo_L && off < row_bytes) {
            /* the request's final partial block: leading bytes of O_n (SP 800-38A 6.5) */
            store_partial(src_row + off, dst_row + off, o[0], o[1], o[2], o[3], row_bytes - off);
        }
    }
}

/* k-iterations [kb0, kb1) of a row, NB blocks per lane at a time */
template <int NB>
__device__ __forceinline__ void ctr_row(uint32_t ybase, const uint4 *rk4, int nr, uint32_t U0, uint32_t U1,
                                        uint32_t U2, uint32_t U3, const uint8_t *src_row, uint8_t *dst_row,
                                        uint32_t lo_L, uint32_t row_bytes, uint32_t lane, uint32_t kb0 = 0,
                                        uint32_t kb1 = 8)
{
    const RowConst rc = row_setup(ybase, rk4, U0, U1, U2, U3, lane);
#pragma unroll 1
    for (uint32_t kb = kb0; kb < kb1; kb += NB) {
        if (kb * 512u >= row_bytes) break;           /* warp-uniform: nothing left in this row  */
        if ((kb + NB) * 32u <= lo_L) continue;       /* warp-uniform: still before the payload  */
        row_blocks<NB>(rc, ybase, rk4, nr, src_row, dst_row, lo_L, row_bytes, lane, kb);
    }
}

/* The counter arithmetic of a request (SP 800-38A B.1 standard incrementing function with m = 128:
 * the counter block is one big-endian integer).  Rows are aligned on the last counter byte being 0. */
struct CtrGeom {
    uint64_t hi, lo_cleared; /* ICB as two big-endian 64-bit halves, last byte cleared */
    uint32_t c0;             /* last byte of the ICB */
};
__device__ __forceinline__ CtrGeom ctr_geom(uint32_t i0, uint32_t i1, uint32_t i2, uint32_t i3)
{
    CtrGeom g;
    g.c0 = i3 >> 24;
    g.hi = ((uint64_t)bswap32(i0) << 32) | bswap32(i1);
    g.lo_cleared = (((uint64_t)bswap32(i2) << 32) | bswap32(i3)) & ~0xffull;
    return g;
}

/* row m of a request of len bytes, k-iterations [kb0, kb1) */
template <int NB>
__device__ __forceinline__ void ctr_request_row(uint32_t ybase, const uint4 *rk4, int nr, const CtrGeom &g,
                                                const uint8_t *src, uint8_t *dst, uint64_t len, uint64_t m,
                                                uint32_t lane, uint32_t kb0 = 0, uint32_t kb1 = 8)
{
    const uint64_t l2 = g.lo_cleared + (m << 8);
    const uint64_t h2 = g.hi + (l2 < g.lo_cleared ? 1ull : 0ull);
    const uint32_t U0 = bswap32((uint32_t)(h2 >> 32)), U1 = bswap32((uint32_t)h2);
    const uint32_t U2 = bswap32((uint32_t)(l2 >> 32)), U3 = bswap32((uint32_t)l2);
    const int64_t row_off = ((int64_t)(m << 8) - (int64_t)g.c0) * 16;
    const int64_t avail = (int64_t)len - row_off;
    const uint32_t row_bytes = avail >= (int64_t)AESOFF_ROW_BYTES ? AESOFF_ROW_BYTES : (uint32_t)avail;
    const uint32_t lo_L = (m == 0) ? g.c0 : 0u;
    ctr_row<NB>(ybase, rk4, nr, U0, U1, U2, U3, src + row_off, dst + row_off, lo_L, row_bytes, lane, kb0, kb1);
}

/* `count` consecutive whole-row units of a request, rows m0, m0 + 1, ...: the first gets the full
 * set-up, the following ones the 10-lookup step unless the increment carries out of counter byte 14. */
template <int NB>
__device__ __forceinline__ void ctr_request_rows(uint32_t ybase, const uint4 *rk4, int nr, const CtrGeom &g,
                                                 const uint8_t *src, uint8_t *dst, uint64_t len, uint64_t m0,
                                                 uint32_t count, uint32_t lane)
{
    RowConst rc;
#pragma unroll 1
    for (uint32_t r = 0; r < count; ++r) {
        const uint64_t m = m0 + r;
        const uint64_t l2 = g.lo_cleared + (m << 8);
        const uint32_t U3 = bswap32((uint32_t)l2);
        if (r == 0 || ((uint32_t)(l2 >> 8) & 0xffu) == 0u) {
            const uint64_t h2 = g.hi + (l2 < g.lo_cleared ? 1ull : 0ull);
            rc = row_setup(ybase, rk4, bswap32((uint32_t)(h2 >> 32)), bswap32((uint32_t)h2), bswap32((uint32_t)(l2 >> 32)),
                           U3, lane);
        } else {
            row_step(rc, ybase, rk4[0].w, U3);
        }
        const int64_t row_off = ((int64_t)(m << 8) - (int64_t)g.c0) * 16;
        const int64_t avail = (int64_t)len - row_off;
        const uint32_t row_bytes = avail >= (int64_t)AESOFF_ROW_BYTES ? AESOFF_ROW_BYTES : (uint32_t)avail;
        const uint32_t lo_L = (m == 0) ? g.c0 : 0u;
#pragma unroll 1
        for (uint32_t kb = 0; kb < 8; kb += NB) {
            if (kb * 512u >= row_bytes) break;
            if ((kb + NB) * 32u <= lo_L) continue;
            row_blocks<NB>(rc, ybase, rk4, nr, src + row_off, dst + row_off, lo_L, row_bytes, lane, kb);
        }
    }
}

/* ------------------------------------------------------------------------------------------ */
/* ECB and CBC-decrypt (SP 800-38A sec. 6.1, 6.2): whole blocks, no counter                     */
/* ------------------------------------------------------------------------------------------ */
/* NB blocks per lane of "row" m (4 KiB of the payload): block L = lane + 32 (kb + b) of the row.
 * MODE: AESOFF_MODE_ECB_ENC  C_j = Cipher(P_j)          (encryption tables, all rounds in full)
 *       AESOFF_MODE_ECB_DEC  P_j = InvCipher(C_j)       (rk4 holds the equivalent inverse cipher's keys)
 *       AESOFF_MODE_CBC_DEC  P_j = InvCipher(C_j) ^ C_{j-1}, C_0 = IV; src and dst must not overlap, since the
 *                            block before this lane's belongs to another lane, warp or CTA                      */
template <int NB, int MODE>
__device__ __forceinline__ void mode_blocks(uint32_t ybase, uint32_t ybd, const uint4 *rk4, int nr, const uint8_t *src_row,
                                            uint8_t *dst_row, uint32_t row_bytes, bool first_row, uint4 iv, uint32_t lane,
                                            uint32_t kb)
{
    uint32_t st[NB][4];
    uint4 prev[NB];
    bool live[NB];
    const uint4 kin = rk4[MODE == AESOFF_MODE_ECB_ENC ? 0 : nr];
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        const uint32_t off = (lane + 32u * (kb + b)) * 16u;
        live[b] = off + 16u <= row_bytes;
        uint4 p = make_uint4(0, 0, 0, 0);
        prev[b] = iv;
        if (live[b]) {
            p = __ldcg(reinterpret_cast<const uint4 *>(src_row + off));
            if (MODE == AESOFF_MODE_CBC_DEC && !(first_row && off == 0u))
                prev[b] = __ldcg(reinterpret_cast<const uint4 *>(src_row + off) - 1);
        }
        st[b][0] = p.x ^ kin.x;
        st[b][1] = p.y ^ kin.y;
        st[b][2] = p.z ^ kin.z;
        st[b][3] = p.w ^ kin.w;
    }
    if (MODE == AESOFF_MODE_ECB_ENC) {
#pragma unroll 1
        for (int r = 1; r < nr; ++r) {
            const uint4 kk = rk4[r];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const uint32_t x0 = st[b][0], x1 = st[b][1], x2 = st[b][2], x3 = st[b][3];
                st[b][0] = TL(0, 0, x0) ^ TL(1, 1, x1) ^ TL(2, 2, x2) ^ TL(3, 3, x3) ^ kk.x;
                st[b][1] = TL(0, 0, x1) ^ TL(1, 1, x2) ^ TL(2, 2, x3) ^ TL(3, 3, x0) ^ kk.y;
                st[b][2] = TL(0, 0, x2) ^ TL(1, 1, x3) ^ TL(2, 2, x0) ^ TL(3, 3, x1) ^ kk.z;
                st[b][3] = TL(0, 0, x3) ^ TL(1, 1, x0) ^ TL(2, 2, x1) ^ TL(3, 3, x2) ^ kk.w;
            }
        }
    } else {
#pragma unroll 1
        for (int r = nr - 1; r > 0; --r) {
            const uint4 kk = rk4[r];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const uint32_t x0 = st[b][0], x1 = st[b][1], x2 = st[b][2], x3 = st[b][3];
                st[b][0] = td_col(x0, x3, x2, x1, ybd) ^ kk.x;
                st[b][1] = td_col(x1, x0, x3, x2, ybd) ^ kk.y;
                st[b][2] = td_col(x2, x1, x0, x3, ybd) ^ kk.z;
                st[b][3] = td_col(x3, x2, x1, x0, ybd) ^ kk.w;
            }
        }
    }
    const uint4 kk = rk4[MODE == AESOFF_MODE_ECB_ENC ? nr : 0];
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        const uint32_t x0 = st[b][0], x1 = st[b][1], x2 = st[b][2], x3 = st[b][3];
        uint4 o;
        if (MODE == AESOFF_MODE_ECB_ENC) {
            o.x = bitsel(bitsel(TL(3, 0, x0), TL(0, 1, x1), 0x000000ffu), bitsel(TL(0, 2, x2), TL(1, 3, x3), 0x00ff0000u), 0x0000ffffu) ^ kk.x;
            o.y = bitsel(bitsel(TL(3, 0, x1), TL(0, 1, x2), 0x000000ffu), bitsel(TL(0, 2, x3), TL(1, 3, x0), 0x00ff0000u), 0x0000ffffu) ^ kk.y;
            o.z = bitsel(bitsel(TL(3, 0, x2), TL(0, 1, x3), 0x000000ffu), bitsel(TL(0, 2, x0), TL(1, 3, x1), 0x00ff0000u), 0x0000ffffu) ^ kk.z;
            o.w = bitsel(bitsel(TL(3, 0, x3), TL(0, 1, x0), 0x000000ffu), bitsel(TL(0, 2, x1), TL(1, 3, x2), 0x00ff0000u), 0x0000ffffu) ^ kk.w;
        } else {
            o.x = tdlast_col(x0, x3, x2, x1, ybd) ^ kk.x;
            o.y = tdlast_col(x1, x0, x3, x2, ybd) ^ kk.y;
            o.z = tdlast_col(x2, x1, x0, x3, ybd) ^ kk.z;
            o.w = tdlast_col(x3, x2, x1, x0, ybd) ^ kk.w;
            if (MODE == AESOFF_MODE_CBC_DEC) {
                o.x ^= prev[b].x;
                o.y ^= prev[b].y;
                o.z ^= prev[b].z;
                o.w ^= prev[b].w;
            }
        }
        if (live[b]) __stcg(reinterpret_cast<uint4 *>(dst_row + (lane + 32u * (kb + b)) * 16u), o);
    }
}

/* rows m0 .. m0 + count - 1 of a request in one of the block modes, k-iterations [kb0, kb1) of each */
template <int NB>
__device__ __noinline__ void mode_request_rows(uint32_t mode, uint32_t ybase, uint32_t ybd, const uint4 *rk4, int nr, uint4 iv,
                                               const uint8_t *src, uint8_t *dst, uint64_t len, uint64_t m0, uint32_t count,
                                               uint32_t lane, uint32_t kb0, uint32_t kb1)
{
#pragma unroll 1
    for (uint32_t r = 0; r < count; ++r) {
        const uint64_t m = m0 + r, row_off = m * AESOFF_ROW_BYTES;
        if (row_off >= len) break;
        const uint32_t row_bytes = len - row_off >= AESOFF_ROW_BYTES ? AESOFF_ROW_BYTES : (uint32_t)(len - row_off);
#pragma unroll 1
        for (uint32_t kb = kb0; kb < kb1; kb += NB) {
            if (kb * 512u >= row_bytes) break;
            if (mode == AESOFF_MODE_ECB_ENC)
                mode_blocks<NB, AESOFF_MODE_ECB_ENC>(ybase, ybd, rk4, nr, src + row_off, dst + row_off, row_bytes, m == 0, iv, lane, kb);
            else if (mode == AESOFF_MODE_ECB_DEC)
                mode_blocks<NB, AESOFF_MODE_ECB_DEC>(ybase, ybd, rk4, nr, src + row_off, dst + row_off, row_bytes, m == 0, iv, lane, kb);
            else
                mode_blocks<NB, AESOFF_MODE_CBC_DEC>(ybase, ybd, rk4, nr, src + row_off, dst + row_off, row_bytes, m == 0, iv, lane, kb);
        }
    }
}

} /* namespace aesoff */
#endif /* AESOFF_CIPHER_CUH */

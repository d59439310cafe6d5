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
 *     per row; per block round 1 is ONE lookup and round 2 FOUR (133 instead of 160 lookups per
 *     AES-128 block, 197 instead of 224 for AES-256).
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

} /* namespace aesoff */
#endif /* AESOFF_CIPHER_CUH */

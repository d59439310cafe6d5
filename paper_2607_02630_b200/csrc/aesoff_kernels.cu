/*
 * aesoff_kernels.cu -- the sm_100a device side of the AES-CTR offload engine.
 *
 * One kernel, `aesoff_engine_kernel`, in two modes:
 *   PERSISTENT  launched once by aes_engine_start(); a dispatcher warp polls the host-mapped
 *               descriptor ring over PCIe and hands chunks to worker groups; lives until
 *               aes_engine_stop().  This is what replaces the paper's "own CUDA stream, polled
 *               by cudaEventQuery" path that is launch-bound at 4 KiB.
 *   DRAIN       the same worker code over a queue the host filled before an ordinary launch
 *               (aes_ctr_launch_batch); exits when the queue is empty.  This is the paper's own
 *               mechanism and the form ncu can replay.
 *
 * The arithmetic (steps a4-a6 of SURVEY.md section 8(a)):
 *   FIPS-197 Cipher() with the SubBytes/ShiftRows/MixColumns of a round folded into four
 *   256-entry word tables (the classical "T-table" form of sec. 5.1: column j of a round's output
 *   is T0[s0,j] ^ T1[s1,j+1] ^ T2[s2,j+2] ^ T3[s3,j+3] ^ roundkey), SP 800-38A sec. 6.5 CTR around it.
 *
 * B200 specifics:
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
#include <cuda_runtime.h>
#include <stdint.h>

#include "aesoff_shared.h"

namespace {

/* ------------------------------------------------------------------------------------------ */
/* shared-memory table layout                                                                  */
/* ------------------------------------------------------------------------------------------ */
constexpr int OFF_T0 = 0;
constexpr int OFF_T1 = 128;
constexpr int OFF_T2 = 65536;
constexpr int OFF_T3 = 65536 + 128;
constexpr uint32_t TABLE_BYTES = 131072;

struct __align__(16) GroupCtl {
    aesoff_dev_desc_t desc;      /* 320 B: descriptor of the request this group last worked on */
    unsigned long long entry;    /* ticket entry handed from the group leader to the group      */
    unsigned long long pad[7];
};                               /* 384 B */
constexpr uint32_t CTRL_BYTES = sizeof(GroupCtl) * AESOFF_GROUPS_PER_CTA;
constexpr unsigned long long ENTRY_EXIT = ~0ull;

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

__device__ __forceinline__ void group_sync(int group)
{
    asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "n"(AESOFF_GROUP_THREADS) : "memory");
}
__device__ __forceinline__ unsigned long long ld_acquire_gpu(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu(unsigned long long *p, unsigned long long v)
{
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_acquire_sys(const volatile uint64_t *p)
{
    unsigned long long v;
    asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t ld_volatile_u32(const volatile uint32_t *p)
{
    uint32_t v;
    asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint4 ld_volatile_v4(const void *p)
{
    uint4 v;
    asm volatile("ld.volatile.global.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "l"(p)
                 : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

/* at most one block per request takes this path, so it is kept out of line */
__device__ __noinline__ void store_partial(const uint8_t *src, uint8_t *dst, uint32_t o0, uint32_t o1, uint32_t o2,
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
/* one row: the (up to) 256 blocks whose counter blocks share bytes 0..14                      */
/* ------------------------------------------------------------------------------------------ */
/* U0..U3   the counter block with its last byte zero, as four little-endian-loaded words
 * rk4      round keys in shared memory (uint4 per round)
 * src_row  address the block with last counter byte 0 would have (may lie before the payload)
 * lo_L     first valid value of the last counter byte in this row (non-zero only in row 0)
 * row_bytes  payload bytes from src_row to the end of the payload, capped at 4096
 * Lane l computes blocks L = l + 32k, k = 0..7, NB at a time.                                  */
template <int NB>
__device__ __forceinline__ void ctr_row(uint32_t ybase, const uint4 *rk4, int nr, uint32_t U0, uint32_t U1,
                                        uint32_t U2, uint32_t U3, const uint8_t *src_row, uint8_t *dst_row,
                                        uint32_t lo_L, uint32_t row_bytes, uint32_t lane)
{
    const uint4 k0 = rk4[0], k1 = rk4[1], k2 = rk4[2];
    /* round 0 (AddRoundKey) on the row's common counter block */
    const uint32_t s0 = U0 ^ k0.x, s1 = U1 ^ k0.y, s2 = U2 ^ k0.z, s3 = U3 ^ k0.w;
    /* round 1: columns 1..3 do not see the last counter byte at all, column 0 sees it through T3 */
    const uint32_t K1_0 = TL(0, 0, s0) ^ TL(1, 1, s1) ^ TL(2, 2, s2) ^ k1.x;
    const uint32_t C1 = TL(0, 0, s1) ^ TL(1, 1, s2) ^ TL(2, 2, s3) ^ TL(3, 3, s0) ^ k1.y;
    const uint32_t C2 = TL(0, 0, s2) ^ TL(1, 1, s3) ^ TL(2, 2, s0) ^ TL(3, 3, s1) ^ k1.z;
    const uint32_t C3 = TL(0, 0, s3) ^ TL(1, 1, s0) ^ TL(2, 2, s1) ^ TL(3, 3, s2) ^ k1.w;
    /* round 2: per column, the three lookups fed by the constant columns C1..C3 */
    const uint32_t K2_0 = TL(1, 1, C1) ^ TL(2, 2, C2) ^ TL(3, 3, C3) ^ k2.x;
    const uint32_t K2_1 = TL(0, 0, C1) ^ TL(1, 1, C2) ^ TL(2, 2, C3) ^ k2.y;
    const uint32_t K2_2 = TL(0, 0, C2) ^ TL(1, 1, C3) ^ TL(3, 3, C1) ^ k2.z;
    const uint32_t K2_3 = TL(0, 0, C3) ^ TL(2, 2, C1) ^ TL(3, 3, C2) ^ k2.w;
    /* address of T3[state byte 15] for last counter byte 0; the byte itself is xored in per block */
    const uint32_t a3 = taddr<3>(s3, ybase) ^ (lane << 8);

#pragma unroll 1
    for (uint32_t kb = 0; kb < 8; kb += NB) {
        if (kb * 512u >= row_bytes) break;           /* warp-uniform: nothing left in this row  */
        if ((kb + NB) * 32u <= lo_L) continue;       /* warp-uniform: still before the payload  */
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
            const uint32_t r1 = K1_0 ^ lds_off<OFF_T3>(a3 ^ ((kb + b) << 13));
            st[b][0] = K2_0 ^ TL(0, 0, r1);
            st[b][1] = K2_1 ^ TL(3, 3, r1);
            st[b][2] = K2_2 ^ TL(2, 2, r1);
            st[b][3] = K2_3 ^ TL(1, 1, r1);
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
        {
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
    }
}

/* ------------------------------------------------------------------------------------------ */
/* one chunk of a request, by one worker group (4 warps; warp w takes rows w, w+4, ...)        */
/* ------------------------------------------------------------------------------------------ */
__device__ __forceinline__ void process_chunk(const GroupCtl *g, uint32_t ybase, uint32_t chunk, uint32_t warp_in_group,
                                              uint32_t lane)
{
    const uint4 *rk4 = reinterpret_cast<const uint4 *>(g->desc.rk);
    const int nr = (int)g->desc.nr;
    const uint64_t len = g->desc.len;
    const uint8_t *src = reinterpret_cast<const uint8_t *>(g->desc.src);
    uint8_t *dst = reinterpret_cast<uint8_t *>(g->desc.dst);
    const uint32_t crows = g->desc.chunk_rows;
    const uint64_t rows = g->desc.rows;
    /* SP 800-38A B.1 standard incrementing function with m = 128: the counter block is a
     * big-endian integer.  c0 = its last byte; rows are aligned on that byte being 0.        */
    const uint32_t i0 = g->desc.icb[0], i1 = g->desc.icb[1], i2 = g->desc.icb[2], i3 = g->desc.icb[3];
    const uint32_t c0 = i3 >> 24;
    const uint64_t hi = ((uint64_t)bswap32(i0) << 32) | bswap32(i1);
    const uint64_t lo_cleared = (((uint64_t)bswap32(i2) << 32) | bswap32(i3)) & ~0xffull;

    const uint64_t row_begin = (uint64_t)chunk * crows;
    uint64_t row_end = row_begin + crows;
    if (row_end > rows) row_end = rows;
    for (uint64_t m = row_begin + warp_in_group; m < row_end; m += AESOFF_GROUP_THREADS / 32) {
        const uint64_t l2 = lo_cleared + (m << 8);
        const uint64_t h2 = hi + (l2 < lo_cleared ? 1ull : 0ull);
        const uint32_t U0 = bswap32((uint32_t)(h2 >> 32)), U1 = bswap32((uint32_t)h2);
        const uint32_t U2 = bswap32((uint32_t)(l2 >> 32)), U3 = bswap32((uint32_t)l2);
        const int64_t row_off = ((int64_t)(m << 8) - (int64_t)c0) * 16;
        const int64_t avail = (int64_t)len - row_off;
        const uint32_t row_bytes = avail >= (int64_t)AESOFF_ROW_BYTES ? AESOFF_ROW_BYTES : (uint32_t)avail;
        const uint32_t lo_L = (m == 0) ? c0 : 0u;
        ctr_row<4>(ybase, rk4, nr, U0, U1, U2, U3, src + row_off, dst + row_off, lo_L, row_bytes, lane);
    }
}

/* ------------------------------------------------------------------------------------------ */
/* worker group: claim a ticket, wait until it is published, process, count down (a3, a7)      */
/* ------------------------------------------------------------------------------------------ */
__device__ void worker_loop(const aesoff_params_t &P, GroupCtl *g, uint32_t ybase, int group, uint32_t gtid)
{
    unsigned long long *g_ticket = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_TICKET);
    unsigned long long *g_published = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_PUBLISHED);
    unsigned long long *g_stop = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_STOP);
    unsigned long long pub_seen = 0;
    unsigned long long cached_seq = 0;
    const uint32_t warp_in_group = gtid >> 5, lane = gtid & 31u;

    for (;;) {
        if (gtid == 0) {
            unsigned long long e = ENTRY_EXIT;
            const unsigned long long t = atomicAdd(g_ticket, 1ull);
            if (P.mode == AESOFF_MODE_DRAIN) {
                if (t < P.drain_total) e = __ldcg(P.tmap + (t & (P.TM - 1)));
            } else {
                bool stop = false;
                while (pub_seen <= t) {
                    pub_seen = ld_acquire_gpu(g_published);
                    if (pub_seen > t) break;
                    if (ld_acquire_gpu(g_stop) != 0) {
                        stop = true;
                        break;
                    }
                    __nanosleep(100);
                }
                if (!stop) e = __ldcg(P.tmap + (t & (P.TM - 1)));
            }
            g->entry = e;
        }
        group_sync(group);
        const unsigned long long e = g->entry;
        if (e == ENTRY_EXIT) break;
        const unsigned long long seq = e >> AESOFF_TICKET_CHUNK_BITS;
        const uint32_t chunk = (uint32_t)(e & ((1u << AESOFF_TICKET_CHUNK_BITS) - 1u));
        const uint32_t slot = (uint32_t)((seq - 1) & (P.R - 1));
        if (seq != cached_seq) {
            /* 320-byte descriptor -> this group's shared memory (20 x 16 B, L2 reads).  Nobody still
             * reads the previous one: every thread has passed the barrier that ended its last chunk. */
            if (gtid < AESOFF_DESC_BYTES / 16) {
                const uint4 v = __ldcg(reinterpret_cast<const uint4 *>(P.dq + slot) + gtid);
                reinterpret_cast<uint4 *>(&g->desc)[gtid] = v;
            }
            cached_seq = seq;
        }
        group_sync(group);
        process_chunk(g, ybase, chunk, warp_in_group, lane);
        group_sync(group); /* all of this chunk's stores are ordered before the leader's fence */
        if (gtid == 0) {
            const uint32_t nchunks = g->desc.nchunks;
            __threadfence();
            const uint32_t d = atomicAdd(P.dq_done + slot, 1u);
            if (d + 1 == nchunks) {
                P.dq_done[slot] = 0;
                __threadfence_system();
                if (P.hmail) P.hmail[slot] = seq;
                *reinterpret_cast<volatile uint64_t *>(P.dev_done_seq + slot) = seq;
            }
        }
    }
}

/* ------------------------------------------------------------------------------------------ */
/* dispatcher warp (persistent mode, CTA 0): host ring -> device queue + tickets  (a3)         */
/* ------------------------------------------------------------------------------------------ */
__device__ void dispatcher_loop(const aesoff_params_t &P, uint32_t lane)
{
    unsigned long long *g_published = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_PUBLISHED);
    unsigned long long *g_stop = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_STOP);
    const uint32_t Rm = P.R - 1;
    unsigned long long next_seq = P.first_seq; /* next sequence number to take from the ring   */
    unsigned long long published = 0;          /* tickets published so far                     */
    unsigned long long oldest = P.first_seq;   /* every seq below this is known to be complete */
    unsigned long long last_activity = globaltimer_ns();

    if (lane == 0) P.hctl[AESOFF_CTL_ALIVE] = 1;

    for (;;) {
        /* phase 1: one PCIe round trip looks at the next 32 slots and at the stop word */
        const unsigned long long s = next_seq + lane;
        const uint32_t slot = (uint32_t)((s - 1) & Rm);
        uint32_t stop = 0;
        const unsigned long long v = ld_acquire_sys(&P.hring[slot].seq);
        if (lane == 0) stop = ld_volatile_u32(P.hctl + AESOFF_CTL_STOP);
        const uint32_t ready = __ballot_sync(0xffffffffu, v == s);
        uint32_t n = __ffs(~ready) - 1; /* length of the ready prefix; 32 if all ready (ffs(0) = 0 -> -1) */
        if (ready == 0xffffffffu) n = 32;
        stop = __shfl_sync(0xffffffffu, stop, 0);
        if (n == 0) {
            bool quit = stop != 0;
            if (!quit && P.idle_exit_ms) {
                const unsigned long long now = globaltimer_ns();
                if (now - last_activity > (unsigned long long)P.idle_exit_ms * 1000000ull) quit = true;
            }
            if (quit) {
                if (lane == 0) {
                    st_release_gpu(g_stop, 1ull);
                    __threadfence_system();
                    P.hctl[AESOFF_CTL_ALIVE] = 2;
                }
                return;
            }
            continue;
        }
        last_activity = globaltimer_ns();

        /* phase 2: second round trip copies the n bodies (18 x 16 B each) into dq */
        for (uint32_t i = lane; i < n * (AESOFF_BODY_BYTES / 16); i += 32) {
            const uint32_t k = i / (AESOFF_BODY_BYTES / 16), j = i % (AESOFF_BODY_BYTES / 16);
            const uint32_t sl = (uint32_t)((next_seq + k - 1) & Rm);
            const uint4 w = ld_volatile_v4(reinterpret_cast<const uint8_t *>(P.hring + sl) + 16 * j);
            reinterpret_cast<uint4 *>(P.dq + sl)[j] = w;
        }
        /* lane k derives the geometry of request next_seq + k */
        uint32_t nchunks = 0, crows = P.chunk_rows;
        unsigned long long rows = 0;
        if (lane < n) {
            const uint4 tail = ld_volatile_v4(reinterpret_cast<const uint8_t *>(P.hring + slot) + 272); /* len, nr, flags */
            const uint32_t icb3 = ld_volatile_u32(reinterpret_cast<const volatile uint32_t *>(P.hring[slot].icb + 3));
            const unsigned long long len = ((unsigned long long)tail.y << 32) | tail.x;
            const unsigned long long nblocks = (len >> 4) + ((len & 15ull) ? 1ull : 0ull);
            const uint32_t c0 = icb3 >> 24;
            rows = nblocks ? ((nblocks + c0 + AESOFF_ROW_BLOCKS - 1) >> 8) : 0ull;
            /* a request must fit the ticket ring with room to spare, and its chunk index 24 bits */
            const unsigned long long max_chunks = P.TM / 4;
            while (((rows + crows - 1) / crows) > max_chunks) crows *= 2;
            nchunks = (uint32_t)((rows + crows - 1) / crows);
        }
        /* exclusive prefix sum of nchunks -> first ticket of each request */
        uint32_t incl = nchunks;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, incl, d);
            if ((int)lane >= d) incl += y;
        }
        /* ticket-ring capacity: every unfinished ticket must stay within TM of the newest.  */
        const unsigned long long first_ticket = published + incl - nchunks;
        for (;;) {
            unsigned long long base = published;
            if (lane == 0) {
                while (oldest < next_seq &&
                       *reinterpret_cast<volatile uint64_t *>(P.dev_done_seq + ((oldest - 1) & Rm)) >= oldest)
                    ++oldest;
                if (oldest < next_seq)
                    base = *reinterpret_cast<volatile uint64_t *>(&P.dq[(oldest - 1) & Rm].pad);
            }
            base = __shfl_sync(0xffffffffu, base, 0);
            const uint32_t fits = __ballot_sync(0xffffffffu, lane >= n || first_ticket + nchunks - base <= P.TM);
            uint32_t nfit = (fits == 0xffffffffu) ? 32u : (uint32_t)(__ffs(~fits) - 1);
            if (nfit > n) nfit = n;
            if (nfit > 0) {
                n = nfit;
                break;
            }
            __nanosleep(200);
        }
        if (lane >= n) nchunks = 0;
        if (lane < n) {
            aesoff_dev_desc_t *d = P.dq + slot;
            d->nchunks = nchunks;
            d->chunk_rows = crows;
            d->seq = s;
            d->rows = rows;
            d->pad = first_ticket;
        }
        /* tickets */
        for (uint32_t k = 0; k < n; ++k) {
            const uint32_t nc = __shfl_sync(0xffffffffu, nchunks, k);
            const unsigned long long ft = __shfl_sync(0xffffffffu, first_ticket, k);
            const unsigned long long sq = next_seq + k;
            for (uint32_t c = lane; c < nc; c += 32)
                P.tmap[(ft + c) & (P.TM - 1)] = (sq << AESOFF_TICKET_CHUNK_BITS) | c;
        }
        const uint32_t total = __shfl_sync(0xffffffffu, incl, n - 1);
        __threadfence();
        __syncwarp();
        published += total;
        if (lane == 0 && total) st_release_gpu(g_published, published);
        /* an empty request (len == 0) has no ticket: complete it here */
        if (lane < n && nchunks == 0) {
            __threadfence_system();
            P.hmail[slot] = s;
            *reinterpret_cast<volatile uint64_t *>(P.dev_done_seq + slot) = s;
        }
        next_seq += n;
    }
}

} /* namespace */

/* ------------------------------------------------------------------------------------------ */
/* the kernel                                                                                  */
/* ------------------------------------------------------------------------------------------ */
__global__ void __launch_bounds__(AESOFF_CTA_THREADS, 1) aesoff_engine_kernel(const aesoff_params_t P)
{
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t tid = threadIdx.x;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem);
    /* tables on a 64 KiB boundary of the shared window so that PRMT can merge base and index */
    const uint32_t tbase = (sbase + 65535u) & ~65535u;
    const uint32_t ctrl = (tbase - sbase >= CTRL_BYTES) ? sbase : tbase + TABLE_BYTES;

    for (uint32_t idx = tid; idx < 256u * 32u; idx += blockDim.x) {
        const uint32_t i = idx >> 5, l = idx & 31u;
        const uint32_t t0 = __ldg(P.T0 + i);
        const uint32_t a = tbase + i * 256u + l * 4u;
        sts(a + OFF_T0, t0);
        sts(a + OFF_T1, rotl32(t0, 8));
        sts(a + OFF_T2, rotl32(t0, 16));
        sts(a + OFF_T3, rotl32(t0, 24));
    }
    if (tid == 0 && blockIdx.x == 0 && P.hctl) P.hctl[AESOFF_CTL_SMEMBASE] = sbase;
    __syncthreads();

    const uint32_t warp = tid >> 5, lane = tid & 31u;
    if (warp == AESOFF_GROUPS_PER_CTA * (AESOFF_GROUP_THREADS / 32)) {
        if (P.mode == AESOFF_MODE_PERSISTENT && blockIdx.x == 0) dispatcher_loop(P, lane);
        return;
    }
    const int group = (int)(warp / (AESOFF_GROUP_THREADS / 32));
    GroupCtl *g = reinterpret_cast<GroupCtl *>(smem + (ctrl - sbase)) + group;
    const uint32_t ybase = tbase | (lane * 4u);
    worker_loop(P, g, ybase, group, tid - group * AESOFF_GROUP_THREADS);
}

/* ------------------------------------------------------------------------------------------ */
/* host-side launch helper (called by aesoff_runtime.cpp)                                      */
/* ------------------------------------------------------------------------------------------ */
extern "C" int aesoff_launch_engine(const aesoff_params_t *params, int n_ctas, void *stream)
{
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(aesoff_engine_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)AESOFF_SMEM_BYTES);
        if (e != cudaSuccess) return (int)e;
        attr_set = true;
    }
    aesoff_engine_kernel<<<n_ctas, AESOFF_CTA_THREADS, AESOFF_SMEM_BYTES, (cudaStream_t)stream>>>(*params);
    return (int)cudaGetLastError();
}

/*
 * aesoff_kernels.cu -- the sm_100a engine kernel of the AES-CTR offload engine.
 *
 * One kernel, `aesoff_engine_kernel`, in two modes:
 *   PERSISTENT  launched once by aes_engine_start(); lives until aes_engine_stop().  This is what
 *               replaces the paper's "own CUDA stream, polled by cudaEventQuery" path that is
 *               launch-bound at 4 KiB.
 *   DRAIN       the same code over a queue the host filled before an ordinary launch
 *               (aes_ctr_launch_batch); exits when the queue is empty.  This is the paper's own
 *               mechanism and the form ncu can replay.
 *
 * Roles inside a CTA (one CTA per SM):
 *   warps 0..15   WORKERS.  A worker claims one *unit* (a 4 KiB row of one request, or 1/8 of a row
 *                 in latency mode) from the CTA's slot queue in shared memory and runs the cipher
 *                 over it (aesoff_cipher.cuh).  Workers never wait on global memory except for the
 *                 payload itself: no barriers, no ticket round trips.
 *   warp 16       SERVICE.  Keeps the CTA's AESOFF_SLOTS slots filled: reserves chunk tickets from
 *                 the device-wide ticket counter, polls them until the dispatcher has written them,
 *                 copies the 96-byte descriptor and the 240-byte expanded key into the slot and opens
 *                 it for claiming -- all while the workers are busy with earlier slots.
 *   warp 17       DISPATCHER (CTA 0, persistent mode only).  Polls the host-mapped descriptor ring
 *                 over PCIe (one round trip per batch of up to 32 requests), expands keys that arrive
 *                 raw (step a1), and cuts each request into chunk tickets (step a3).
 * Completion (step a7): the worker that finishes the last unit of a slot counts the request's chunks
 * down in global memory; the last chunk's finisher fences at system scope and writes the request's
 * sequence number into the host-mapped mailbox.
 */
#include <cuda_runtime.h>
#include <stdint.h>

#include "aesoff_cipher.cuh"
#include "aesoff_shared.h"

using namespace aesoff;

namespace {

constexpr uint32_t AESOFF_STAGE_STRIDE = 36; /* words per staged descriptor: 32 + padding against bank conflicts */

/* ------------------------------------------------------------------------------------------ */
/* per-CTA control block in shared memory                                                      */
/* ------------------------------------------------------------------------------------------ */
struct __align__(16) Slot {
    aesoff_dev_desc_t desc; /*  96 B: descriptor of the request                                 */
    uint4 rk4[16];          /* 256 B: its expanded key (ktab entry), one uint4 per round        */
    uint32_t unit0_row;     /* first row of this chunk                                          */
    uint32_t ring_slot;     /* index of the request in dq / mailbox                             */
    uint32_t n_units;
    uint32_t n_rows;        /* rows of this chunk                                               */
    uint32_t pad_[3];
    uint32_t fine;          /* unit size: 0 rows (AESOFF_ROWS_PER_UNIT of them), AESOFF_FLAG_HALF half a row (128 blocks),
                               AESOFF_FLAG_FINE one k-iteration of a row (32 blocks)            */
};                          /* 384 B */

struct __align__(16) CtaCtl {
    Slot slot[AESOFF_SLOTS];
    /* claim[s] = n_units << 16 | next unit.  Written whole by the service warp when it opens the
     * slot (after the descriptor), incremented by claiming workers: one atomic snapshot tells a
     * worker both the unit it got and whether that unit exists.                                 */
    uint32_t claim[AESOFF_SLOTS];
    uint32_t done[AESOFF_SLOTS];  /* units finished                                              */
    uint32_t stamp[AESOFF_SLOTS]; /* fill order, so that workers take the oldest open slot first */
    uint32_t busy[AESOFF_SLOTS];  /* 0 free, 1 filled and not yet completed                      */
    uint32_t exit_flag;
    uint32_t pad[3];
    /* dispatcher (CTA 0): the descriptors of one poll, as read from the host ring */
    uint32_t stage[32][AESOFF_STAGE_STRIDE];
};
constexpr uint32_t CTRL_BYTES = sizeof(CtaCtl);
constexpr uint32_t CLAIM_EXIT = 0xffffffffu;
static_assert(CTRL_BYTES <= 32u * 1024u, "control block must fit beside the tables (AESOFF_SMEM_BYTES)");

__device__ __forceinline__ uint32_t lds_volatile(const uint32_t *p)
{
    uint32_t v;
    asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"((uint32_t)__cvta_generic_to_shared(p)) : "memory");
    return v;
}
__device__ __forceinline__ void sts_volatile(uint32_t *p, uint32_t v)
{
    asm volatile("st.volatile.shared.u32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(p)), "r"(v) : "memory");
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

/* ------------------------------------------------------------------------------------------ */
/* worker warp (steps a4-a7)                                                                   */
/* ------------------------------------------------------------------------------------------ */
/* Takes a unit of the oldest open slot.  Returns slot << 16 | unit, or CLAIM_EXIT.             */
__device__ __forceinline__ uint32_t claim_unit(CtaCtl *c, uint32_t lane)
{
    uint32_t backoff = 32u;
    for (;;) {
        uint32_t w = 0, st = 0;
        if (lane < AESOFF_SLOTS) {
            w = lds_volatile(&c->claim[lane]);
            st = lds_volatile(&c->stamp[lane]);
        }
        const uint32_t avail = __ballot_sync(0xffffffffu, (w & 0xffffu) < (w >> 16));
        if (avail) {
            /* oldest first; live stamps lie within AESOFF_SLOTS of each other, so the signed
             * distance to any live one orders them even when the counter wraps                  */
            const uint32_t ref = __shfl_sync(0xffffffffu, st, __ffs(avail) - 1);
            uint32_t key = 0xffffffffu;
            if ((avail >> lane) & 1u) key = ((st - ref + 0x1000u) << 5) | lane;
            const uint32_t s = __reduce_min_sync(0xffffffffu, key) & 31u;
            uint32_t v = 0;
            if (lane == 0) v = atomicAdd(&c->claim[s], 1u);
            if (lane == 0) __threadfence_block(); /* acquire side of the service warp's slot publication */
            v = __shfl_sync(0xffffffffu, v, 0);
            __syncwarp();
            if ((v & 0xffffu) < (v >> 16)) return (s << 16) | (v & 0xffffu);
            continue;
        }
        if (lds_volatile(&c->exit_flag)) return CLAIM_EXIT;
        /* an idle worker's polling runs on the very pipe the busy ones are bound by: back off */
        __nanosleep(backoff);
        if (backoff < 256u) backoff <<= 1;
    }
}

/* The slot's chunk is finished: count the request's chunks down; the last one signals the host. */
__device__ __forceinline__ void complete_chunk(const aesoff_params_t &P, CtaCtl *c, uint32_t s)
{
    const Slot *sl = &c->slot[s];
    const uint32_t ring = sl->ring_slot, nchunks = sl->desc.nchunks;
    const unsigned long long seq = sl->desc.seq;
    /* the other workers' stores to dst happen-before their done-count increments (fence.cta +
     * shared-memory atomic), which this thread has observed: this fence is cumulative over them */
    __threadfence();
    bool last = true;
    if (nchunks > 1) {
        const uint32_t d = atomicAdd(P.dq_done + ring, 1u);
        last = (d + 1 == nchunks);
        if (last) P.dq_done[ring] = 0;
    }
    if (last) {
        __threadfence_system();
        if (P.hmail) P.hmail[ring] = seq;
        *reinterpret_cast<volatile uint64_t *>(P.dev_done_seq + ring) = seq;
    }
    sts_volatile(&c->busy[s], 0u); /* the service warp may refill the slot */
}

__device__ void worker_loop(const aesoff_params_t &P, CtaCtl *c, uint32_t ybase, uint32_t lane)
{
#ifdef AESOFF_DEBUG
    bool first = true;
#endif
    for (;;) {
        const uint32_t got = claim_unit(c, lane);
        if (got == CLAIM_EXIT) break;
#ifdef AESOFF_DEBUG
        if (lane == 0 && first) {
            atomicMin(reinterpret_cast<unsigned long long *>(P.counters) + 20 + 3, globaltimer_ns()); /* first unit claimed anywhere */
            atomicMax(reinterpret_cast<unsigned long long *>(P.counters) + 20 + 4, globaltimer_ns()); /* last warp gets its first unit */
        }
        first = false;
#endif
        const uint32_t s = got >> 16, u = got & 0xffffu;
        const Slot *sl = &c->slot[s];
        const uint4 *rk4 = sl->rk4;
        const int nr = (int)sl->desc.nr;
        const uint64_t len = sl->desc.len;
        const uint8_t *src = reinterpret_cast<const uint8_t *>(sl->desc.src);
        uint8_t *dst = reinterpret_cast<uint8_t *>(sl->desc.dst);
        const CtrGeom g = ctr_geom(sl->desc.icb[0], sl->desc.icb[1], sl->desc.icb[2], sl->desc.icb[3]);
        const uint32_t n_units = sl->n_units;
        const uint32_t fine = sl->fine;
        if (fine & AESOFF_FLAG_FINE) {
            const uint64_t m = (uint64_t)sl->unit0_row + (u >> 3);
            ctr_request_row<1>(ybase, rk4, nr, g, src, dst, len, m, lane, u & 7u, (u & 7u) + 1u);
        } else if (fine & AESOFF_FLAG_HALF) {
            const uint64_t m = (uint64_t)sl->unit0_row + (u >> 1);
            ctr_request_row<4>(ybase, rk4, nr, g, src, dst, len, m, lane, (u & 1u) * 4u, (u & 1u) * 4u + 4u);
        } else {
            /* a whole-row unit is AESOFF_ROWS_PER_UNIT consecutive rows: half the claims and done counts,
             * and the second row's set-up is a 10-lookup step from the first's */
            const uint32_t first = u * AESOFF_ROWS_PER_UNIT, crows_here = sl->n_rows;
            const uint32_t cnt = crows_here - first < AESOFF_ROWS_PER_UNIT ? crows_here - first : AESOFF_ROWS_PER_UNIT;
            ctr_request_rows<AESOFF_NB>(ybase, rk4, nr, g, src, dst, len, (uint64_t)sl->unit0_row + first, cnt, lane);
        }
        __syncwarp();
        if (lane == 0) {
            __threadfence_block();
            const uint32_t d = atomicAdd(&c->done[s], 1u);
            if (d + 1 == n_units) complete_chunk(P, c, s);
        }
        __syncwarp();
    }
}

/* ------------------------------------------------------------------------------------------ */
/* service warp: global ticket queue -> this CTA's slots, ahead of the workers  (a3)           */
/* ------------------------------------------------------------------------------------------ */
/* Lane j < AESOFF_SLOTS owns slot j.  All lanes run in lock step; nothing here is on the
 * workers' critical path as long as at least one slot is open.                                 */
__device__ void service_loop(const aesoff_params_t &P, CtaCtl *c, uint32_t lane)
{
    unsigned long long *g_ticket = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_TICKET);
    const bool persistent = (P.mode == AESOFF_MODE_PERSISTENT);
    const bool mine = lane < AESOFF_SLOTS;
    unsigned long long *g_idle = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_IDLE);
    bool have = false;          /* this lane holds a reserved ticket for its (free) slot */
    unsigned long long t = 0;   /* that ticket */
    uint32_t stamp_base = 0;
    bool counted_idle = false;  /* this CTA is included in the device-wide idle-CTA count */

    for (;;) {
        const bool is_free = mine && lds_volatile(&c->busy[lane]) == 0u;
        const uint32_t busy_mask = __ballot_sync(0xffffffffu, mine && !is_free);
        const uint32_t have_mask = __ballot_sync(0xffffffffu, have);
        uint32_t need = __ballot_sync(0xffffffffu, is_free && !have);
        if (persistent && (busy_mask == 0u) != counted_idle) {
            /* the dispatcher cuts requests fine only while a good part of the GPU has nothing to do */
            counted_idle = !counted_idle;
            if (lane == 0) atomicAdd(g_idle, counted_idle ? 1ull : ~0ull);
        }

        /* two independent L2 reads, issued back to back.  (a) The tickets this warp holds: a ticket
         * is one self-validating 16-byte word, so polling it finds out that it exists and fetches
         * it in the same access.  (b) Ticket counter and published count, one 16-byte word.       */
        if (!persistent && have && t >= P.drain_total) have = false; /* reserved past the end of the queue */
        const bool polled = have;
        uint4 tv = make_uint4(0, 0, 0, 0);
        if (polled) tv = ld_volatile_v4(P.tmap + (t & (unsigned long long)(P.TM - 1)));
        unsigned long long tk = 0, pub = 0;
        if (lane == 0) {
            const uint4 v = ld_volatile_v4(g_ticket);
            tk = ((unsigned long long)v.y << 32) | v.x;
            pub = ((unsigned long long)v.w << 32) | v.z;
        }
        tk = __shfl_sync(0xffffffffu, tk, 0);
        pub = __shfl_sync(0xffffffffu, pub, 0);

        /* 1. reserve tickets: as many as are visibly waiting, capped by the free slots.  An idle
         *    CTA of the persistent engine also keeps ONE reservation on a ticket that does not
         *    exist yet, so that a lone request finds 148 CTAs waiting, one ticket each.         */
        unsigned long long avail = pub > tk ? pub - tk : 0ull;
        if (persistent && busy_mask == 0u && have_mask == 0u && avail == 0ull) avail = 1ull;
        /*    A CTA does not hoard: what it holds (unclaimed units of its open slots plus the tickets
         *    it has reserved, in 1/8-row units) stays near one and a half rows per worker -- enough
         *    to hide a refill (microseconds against 10 us per row), little enough that the end of a
         *    burst is not left to the few CTAs that grabbed 16 chunks each.                        */
        {
            const uint32_t per_ticket = P.chunk_rows * 8u;
            uint32_t held = 0;
            if (mine && !is_free) {
                const uint32_t w = lds_volatile(&c->claim[lane]);
                const uint32_t left = (w >> 16) > (w & 0xffffu) ? (w >> 16) - (w & 0xffffu) : 0u;
                const uint32_t f = c->slot[lane].fine;
                held = (f & AESOFF_FLAG_FINE) ? left : (f & AESOFF_FLAG_HALF) ? left * 4u : left * 8u * AESOFF_ROWS_PER_UNIT;
            } else if (have) {
                held = per_ticket;
            }
            held = __reduce_add_sync(0xffffffffu, held);
            const uint32_t hold_max = AESOFF_WORKER_WARPS * 12u; /* 1.5 rows per worker */
            unsigned long long cap = held < hold_max ? (hold_max - held + per_ticket - 1u) / per_ticket : 0u;
            if (cap == 0ull && busy_mask == 0u && have_mask == 0u) cap = 1ull;
            /* ... nor takes more than its share of a short queue: the last tickets of a burst (and the
             * tickets of a lone request) spread over all CTAs instead of piling up on the first few  */
            const uint32_t a32 = avail > 0x100000ull ? 0x100000u : (uint32_t)avail; /* 32-bit division */
            const uint32_t share = (a32 + gridDim.x - 1u) / gridDim.x;
            if (cap > share) cap = share ? share : 1ull;
            if (avail > cap) avail = cap;
        }
        uint32_t n_need = __popc(need);
        if ((unsigned long long)n_need > avail) {
            n_need = (uint32_t)avail;
            need = n_need ? (need & ((2u << (__fns(need, 0, n_need) & 31)) - 1u)) : 0u; /* lowest n_need bits set in need */
        }
        if (need) {
            unsigned long long base = 0;
            if (lane == 0) base = atomicAdd(g_ticket, (unsigned long long)n_need);
            base = __shfl_sync(0xffffffffu, base, 0);
            if ((need >> lane) & 1u) {
                t = base + __popc(need & ((1u << lane) - 1u));
                have = true;
            }
        }

        /* 2. tickets that have been published by now */
        const bool ready = polled && tv.w == (uint32_t)t + 1u;
        const uint32_t ready_mask = __ballot_sync(0xffffffffu, ready);
        if (ready_mask) {
            /* The expanded key is ordered before the ticket by the dispatcher's fence (only requests that
             * brought a raw key pay for one); the descriptor is not: its 8 pieces carry the request's
             * sequence number and a piece read too early is simply read again.                          */
            __threadfence();
            const uint32_t seq32 = tv.x, chunk = tv.y & AESOFF_TICKET_CHUNK_MASK, keyloc = tv.z;
            const uint32_t ring = (seq32 - 1u) & (P.R - 1u);
            const uint32_t unit_mode = tv.y >> AESOFF_TICKET_MODE_SHIFT; /* AESOFF_FLAG_FINE / _HALF / 0 */
            /* descriptor pieces (lanes 0..7) and expanded key (lanes 8..22), 16 B each; four slots' loads are
             * in flight together (one L2 round trip per four slots, not per slot)                        */
            for (uint32_t m = ready_mask; m;) {
                uint32_t sj[4];
                uint4 v[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    sj[q] = 32u;
                    if (m) {
                        sj[q] = __ffs(m) - 1;
                        m &= m - 1u;
                    }
                }
                for (;;) {
                    bool stale = false;
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        if (sj[q] < 32u) {
                            const uint32_t rj = __shfl_sync(0xffffffffu, ring, sj[q]);
                            const uint32_t kj = __shfl_sync(0xffffffffu, keyloc, sj[q]);
                            if (lane < 8)
                                v[q] = ld_volatile_v4(reinterpret_cast<const uint4 *>(P.dq + rj) + lane);
                            else if (lane < 8 + 15)
                                v[q] = __ldcg(reinterpret_cast<const uint4 *>(P.ktab + kj) + (lane - 8));
                        }
                    }
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        if (sj[q] < 32u) {
                            const uint32_t want = __shfl_sync(0xffffffffu, seq32, sj[q]);
                            if (lane < 8 && v[q].w != want) stale = true;
                        }
                    }
                    if (!__any_sync(0xffffffffu, stale)) break;
                }
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    if (sj[q] < 32u) {
                        if (lane < 8) {
                            uint32_t *dw = reinterpret_cast<uint32_t *>(&c->slot[sj[q]].desc) + 3u * lane;
                            dw[0] = v[q].x;
                            dw[1] = v[q].y;
                            dw[2] = v[q].z;
                        } else if (lane < 8 + 15) {
                            c->slot[sj[q]].rk4[lane - 8] = v[q];
                        }
                    }
                }
            }
            __syncwarp();
            if (ready) {
                Slot *sl = &c->slot[lane];
                const unsigned long long rows = sl->desc.rows;
                const uint32_t crows = sl->desc.chunk_rows;
                const unsigned long long row0 = (unsigned long long)chunk * crows;
                const uint32_t nrows = (uint32_t)((rows - row0) < crows ? (rows - row0) : crows);
                const uint32_t fine = unit_mode & (AESOFF_FLAG_FINE | AESOFF_FLAG_HALF);
                const uint32_t n_units = (fine & AESOFF_FLAG_FINE) ? nrows * 8u : (fine & AESOFF_FLAG_HALF) ? nrows * 2u
                                         : (nrows + AESOFF_ROWS_PER_UNIT - 1u) / AESOFF_ROWS_PER_UNIT;
                sl->n_rows = nrows;
                sl->unit0_row = (uint32_t)row0;
                sl->ring_slot = ring;
                sl->n_units = n_units;
                sl->fine = fine;
                c->done[lane] = 0u;
                c->stamp[lane] = stamp_base + __popc(ready_mask & ((1u << lane) - 1u));
                c->busy[lane] = 1u;
                __threadfence_block();
                sts_volatile(&c->claim[lane], n_units << 16); /* open the slot */
                have = false;
            }
            stamp_base += __popc(ready_mask);
            continue;
        }

        /* 3. nothing to load: time to leave? */
        if (!persistent) {
            if (tk >= P.drain_total && busy_mask == 0u && __ballot_sync(0xffffffffu, have) == 0u) break;
        } else if (busy_mask == 0u) {
            unsigned long long stop = 0;
            if (lane == 0) stop = ld_acquire_gpu(reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_STOP));
            if (__shfl_sync(0xffffffffu, stop, 0) != 0ull) break;
        }
        if (!need) __nanosleep(100);
    }
    if (lane == 0) sts_volatile(&c->exit_flag, 1u);
}

/* ------------------------------------------------------------------------------------------ */
/* dispatcher warp (persistent mode, CTA 0): host ring -> device queue + tickets  (a3)         */
/* ------------------------------------------------------------------------------------------ */
/* One iteration = ONE PCIe round trip: the warp reads the next 8 (quiet) or 32 (busy) ring slots,
 * 128 B each, as 16-byte pieces that validate themselves (aesoff_shared.h), so there is no
 * flag-then-body dependency.  Everything after that is on-chip or L2: geometry, key expansion
 * for raw keys, descriptor and ticket stores, one release of the published count.             */
__device__ void dispatcher_loop(const aesoff_params_t &P, CtaCtl *c, uint32_t ybase, uint32_t lane)
{
    unsigned long long *g_idle = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_IDLE);
    unsigned long long *g_published = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_PUBLISHED);
    unsigned long long *g_stop = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_STOP);
    const uint32_t Rm = P.R - 1;
    unsigned long long next_seq = P.first_seq; /* next sequence number to take from the ring   */
    unsigned long long published = 0;          /* tickets published so far                     */
    unsigned long long oldest = P.first_seq;   /* every seq below this is known to be complete */
    unsigned long long base = 0;               /* first ticket of request `oldest` at the last scan */
    unsigned long long last_activity = globaltimer_ns();
    uint32_t wide = 0;                         /* 0: poll 8 slots, 1: poll 32                  */
    uint32_t n_eighths = 0, n_halves = 0, n_rows = 0;
    bool stats_dirty = false;

    if (lane == 0) P.hctl[AESOFF_CTL_ALIVE] = 1;

    /* One poll = the next 8 (quiet) or 32 (busy) ring slots as 16-byte pieces, plus the stop word and two
     * device counters.  piece g = 32 j + lane: slot g / 8 after the poll's first sequence number, piece g % 8.
     * A poll is issued as soon as the previous one has been looked at, i.e. BEFORE that batch is processed:
     * the PCIe round trip of the next batch runs under the on-chip work of this one.                       */
    uint4 pc[8];
    uint32_t p_stop = 0, p_nload = 2u;
    unsigned long long p_idle = 0, p_reserved = 0;
#define ISSUE_POLL(seq0)                                                                                     \
    do {                                                                                                     \
        p_nload = wide ? 8u : 2u;                                                                            \
        _Pragma("unroll") for (uint32_t j = 0; j < 8; ++j)                                                  \
        {                                                                                                    \
            pc[j] = make_uint4(0, 0, 0, 0);                                                                  \
            if (j < p_nload) {                                                                               \
                const uint32_t k_ = j * 4u + (lane >> 3);                                                    \
                const uint32_t sl_ = (uint32_t)(((seq0) + k_ - 1) & Rm);                                     \
                pc[j] = ld_volatile_v4(reinterpret_cast<const uint8_t *>(P.hring + sl_) + 16u * (lane & 7u)); \
            }                                                                                                \
        }                                                                                                    \
        if (lane == 0) {                                                                                     \
            p_stop = ld_volatile_u32(P.hctl + AESOFF_CTL_STOP);                                              \
            p_idle = *reinterpret_cast<volatile unsigned long long *>(g_idle);                               \
            p_reserved = *reinterpret_cast<volatile unsigned long long *>(P.counters + AESOFF_CNT_TICKET);   \
        }                                                                                                    \
    } while (0)
    bool repoll = true; /* the poll in flight (if any) does not start at next_seq */

    for (;;) {
        /* ---- phase 1: the PCIe round trip ---------------------------------------------------- */
        if (repoll) ISSUE_POLL(next_seq);
        repoll = false;
        const uint32_t nload = p_nload;
        uint32_t stop = p_stop;
        unsigned long long idle = p_idle, reserved = p_reserved;
#pragma unroll
        for (uint32_t j = 0; j < 8; ++j) {
            if (j < nload) {
                const uint32_t k = j * 4u + (lane >> 3);
                *reinterpret_cast<uint4 *>(&c->stage[k][4u * (lane & 7u)]) = pc[j];
            }
        }
        __syncwarp();
        /* lane k looks at slot k of the poll */
        const unsigned long long s = next_seq + lane;
        const uint32_t slot = (uint32_t)((s - 1) & Rm);
        const uint32_t *sw = c->stage[lane];
        const uint32_t tag = (uint32_t)s;
        uint32_t kw = 0;
        bool valid = false;
        if (lane < nload * 4u) {
            kw = sw[AESOFF_PW_INDEX(AESOFF_PW_KEY)];
            valid = sw[3] == tag && sw[7] == tag && sw[11] == tag && sw[15] == tag;
            if (valid && (kw & AESOFF_KW_RAW))
                valid = sw[19] == tag && sw[23] == tag && sw[27] == tag && sw[31] == tag;
        }
        const uint32_t vmask = __ballot_sync(0xffffffffu, valid);
        uint32_t n = (vmask == 0xffffffffu) ? 32u : (uint32_t)(__ffs(~vmask) - 1); /* length of the ready prefix */
        stop = __shfl_sync(0xffffffffu, stop, 0);
        idle = __shfl_sync(0xffffffffu, idle, 0);
        reserved = __shfl_sync(0xffffffffu, reserved, 0);
        wide = (n >= 8u) ? 1u : 0u;
        const uint32_t n_seen = n;
        if (n != 0) ISSUE_POLL(next_seq + n); /* the staged copy of this poll is in shared memory: pc[] is free */
        if (n == 0) {
            repoll = true;
            if (stats_dirty) {
                /* not on a request's way: a PCIe write in flight would hold up the next fence */
                if (lane == 0) {
                    P.hctl[AESOFF_CTL_CUT_EIGHTHS] = n_eighths;
                    P.hctl[AESOFF_CTL_CUT_HALVES] = n_halves;
                    P.hctl[AESOFF_CTL_CUT_ROWS] = n_rows;
                }
                stats_dirty = false;
            }
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

        /* ---- phase 2: lane k derives the geometry of request next_seq + k ---------------------- */
        unsigned long long len = 0, rows = 0;
        uint32_t nchunks = 0, crows = P.chunk_rows, fine = 0, nr = 0;
        /* Latency modes.  A request of up to 64 KiB is always cut into 1/8-row units (32 blocks per
         * warp; it is submission-bound anyway).  A larger one, up to fine_rows rows, is cut by the
         * load it meets = rows not yet reserved by any CTA + the rows of this poll up to and including it:
         *   - 1/8-row units while a quarter of the CTAs have nothing to do and the load makes at most two
         *     waves of such units over the GPU's worker warps (a lone request: spread it over every
         *     warp; 17 % more lookups per block, nobody is waiting for them);
         *   - half rows while the load makes at most one and a half waves of half rows: half the time
         *     per unit for 2.5 % more lookups;
         *   - whole rows otherwise (saturation).                                                     */
        const unsigned long long backlog = published > reserved ? published - reserved : 0ull;
        const bool gpu_idle = idle * 4ull >= (unsigned long long)gridDim.x;
        const unsigned long long warps = (unsigned long long)gridDim.x * AESOFF_WORKER_WARPS;
        if (lane < n) {
#define PW(p) sw[AESOFF_PW_INDEX(p)]
            /* only what the geometry needs; the rest goes from the staging area straight into dq */
            len = ((unsigned long long)PW(AESOFF_PW_LEN + 1) << 32) | PW(AESOFF_PW_LEN);
            nr = kw >> 24;
            const unsigned long long nblocks = (len >> 4) + ((len & 15ull) ? 1ull : 0ull);
            const uint32_t c0 = PW(AESOFF_PW_ICB + 3) >> 24;
            rows = nblocks ? ((nblocks + c0 + AESOFF_ROW_BLOCKS - 1) >> 8) : 0ull;
        }
        /* rows of this poll up to and including request k */
        unsigned long long rows_incl = (lane < n) ? rows : 0ull;
        if (n > 1) { /* a lone request (the latency case) skips the scan */
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned long long y = __shfl_up_sync(0xffffffffu, rows_incl, d);
                if ((int)lane >= d) rows_incl += y;
            }
        }
        if (lane < n) {
            const unsigned long long load = backlog * P.chunk_rows + rows_incl;
            if (P.fine_rows && rows <= P.fine_rows) {
                if (rows <= AESOFF_FINE_ALWAYS_ROWS || (gpu_idle && load * 8ull <= 2ull * warps)) {
                    fine = AESOFF_FLAG_FINE;
                    crows = crows > 1u ? crows / 2u : 1u;
                } else if (load * 4ull <= 3ull * warps) {
                    fine = AESOFF_FLAG_HALF;
                }
            }
            /* a request must fit the ticket ring with room to spare */
            const unsigned long long max_chunks = P.TM / 4;
            while (((rows + crows - 1) / crows) > max_chunks) crows *= 2;
            nchunks = (uint32_t)((rows + crows - 1) / crows);
        }
        /* exclusive prefix sum of nchunks -> first ticket of each request */
        uint32_t incl = nchunks;
        if (n > 1) {
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t y = __shfl_up_sync(0xffffffffu, incl, d);
                if ((int)lane >= d) incl += y;
            }
        }
        const unsigned long long first_ticket = published + incl - nchunks;
        /* ticket-ring capacity: every unfinished ticket must stay within TM of the newest.  `base`
         * is only refreshed (32 completion words per L2 round trip) when the cached one says no. */
        for (;;) {
            const uint32_t fits = __ballot_sync(0xffffffffu, lane >= n || first_ticket + nchunks - base <= P.TM);
            uint32_t nfit = (fits == 0xffffffffu) ? 32u : (uint32_t)(__ffs(~fits) - 1);
            if (nfit > n) nfit = n;
            if (nfit == n) break;
            for (;;) {
                const unsigned long long q = oldest + lane;
                bool fin = false;
                if (q < next_seq)
                    fin = *reinterpret_cast<volatile uint64_t *>(P.dev_done_seq + ((q - 1) & Rm)) >= q;
                const uint32_t fm = __ballot_sync(0xffffffffu, fin);
                const uint32_t adv = (fm == 0xffffffffu) ? 32u : (uint32_t)(__ffs(~fm) - 1);
                oldest += adv;
                if (adv < 32u) break;
            }
            unsigned long long nb = published;
            if (lane == 0 && oldest < next_seq)
                nb = *reinterpret_cast<volatile uint64_t *>(&P.dq[(oldest - 1) & Rm].w[24]); /* first_ticket: words 18, 19 */
            nb = __shfl_sync(0xffffffffu, nb, 0);
            if (nb == base) {
                if (nfit > 0) {
                    n = nfit;
                    break;
                }
                __nanosleep(200);
            }
            base = nb;
        }
        if (lane >= n) nchunks = 0;
        if (n != n_seen) repoll = true; /* the ticket ring took fewer requests than the poll in flight assumes */
        {   /* statistics for aes_engine_info */
            const uint32_t me = __ballot_sync(0xffffffffu, lane < n && (fine & AESOFF_FLAG_FINE));
            const uint32_t mh = __ballot_sync(0xffffffffu, lane < n && (fine & AESOFF_FLAG_HALF));
            n_eighths += __popc(me);
            n_halves += __popc(mh);
            n_rows += n - __popc(me) - __popc(mh);
            stats_dirty = true; /* written to the host when the ring is next found empty */
        }

        /* ---- phase 3: keys, descriptors, tickets ----------------------------------------------- */
        uint32_t keyloc = kw & 0xffffu;
        if (!(kw & AESOFF_KW_RAW) && keyloc >= AESOFF_KEY_IDS) keyloc = AESOFF_KEY_IDS + slot; /* never sent by the host */
        if (lane < n && (kw & AESOFF_KW_RAW)) {
            if (!(kw & AESOFF_KW_INSTALL) || keyloc >= AESOFF_KEY_IDS) keyloc = AESOFF_KEY_IDS + slot;
            uint32_t key[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) key[i] = PW(AESOFF_PW_RAWKEY + i);
            if (nr == 10)
                key_expand<4>(ybase, key, P.ktab[keyloc].rk); /* step a1 on the device */
            else if (nr == 12)
                key_expand<6>(ybase, key, P.ktab[keyloc].rk);
            else
                key_expand<8>(ybase, key, P.ktab[keyloc].rk);
        }
        if (lane < n) {
            /* the 24 descriptor words as 8 pieces of {3 words, tag}: see aesoff_dq_entry_t */
            uint4 *d4 = reinterpret_cast<uint4 *>(P.dq + slot);
            const uint32_t tg = (uint32_t)s;
            d4[0] = make_uint4(PW(AESOFF_PW_ICB + 0), PW(AESOFF_PW_ICB + 1), PW(AESOFF_PW_ICB + 2), tg);
            d4[1] = make_uint4(PW(AESOFF_PW_ICB + 3), PW(AESOFF_PW_SRC), PW(AESOFF_PW_SRC + 1), tg);
            d4[2] = make_uint4(PW(AESOFF_PW_DST), PW(AESOFF_PW_DST + 1), (uint32_t)len, tg);
            d4[3] = make_uint4((uint32_t)(len >> 32), nr, fine, tg);
            d4[4] = make_uint4(nchunks, crows, (uint32_t)s, tg);
            d4[5] = make_uint4((uint32_t)(s >> 32), (uint32_t)rows, (uint32_t)(rows >> 32), tg);
            d4[6] = make_uint4((uint32_t)first_ticket, (uint32_t)(first_ticket >> 32), keyloc, tg);
            d4[7] = make_uint4(0u, 0u, 0u, tg);
        }
#undef PW
        /* expanded keys (if any request of this poll brought a raw one) before the tickets that point at
         * them; descriptors need no fence, their pieces validate themselves */
        if (__any_sync(0xffffffffu, lane < n && (kw & AESOFF_KW_RAW))) __threadfence();
        __syncwarp();
        /* a request of up to eight chunks (the fine-grained regime: every request of the poll) gets its
         * tickets from its own lane; the warp then shares out the long ones, 32 tickets per step */
        if (lane < n) {
            const uint32_t md = fine << AESOFF_TICKET_MODE_SHIFT;
            for (uint32_t ch = 0; ch < nchunks && ch < 8u; ++ch) {
                const unsigned long long tno = first_ticket + ch;
                *reinterpret_cast<uint4 *>(P.tmap + (tno & (unsigned long long)(P.TM - 1))) =
                    make_uint4((uint32_t)s, ch | md, keyloc, (uint32_t)tno + 1u);
            }
        }
        for (uint32_t big = __ballot_sync(0xffffffffu, lane < n && nchunks > 8u); big; big &= big - 1u) {
            const uint32_t k = __ffs(big) - 1;
            const uint32_t nc = __shfl_sync(0xffffffffu, nchunks, k);
            const unsigned long long ft = __shfl_sync(0xffffffffu, first_ticket, k);
            const uint32_t kl = __shfl_sync(0xffffffffu, keyloc, k);
            const uint32_t md = __shfl_sync(0xffffffffu, fine, k) << AESOFF_TICKET_MODE_SHIFT;
            const uint32_t sq = (uint32_t)(next_seq + k);
            for (uint32_t ch = 8u + lane; ch < nc; ch += 32) {
                const unsigned long long tno = ft + ch;
                *reinterpret_cast<uint4 *>(P.tmap + (tno & (unsigned long long)(P.TM - 1))) =
                    make_uint4(sq, ch | md, kl, (uint32_t)tno + 1u);
            }
        }
        const uint32_t total = __shfl_sync(0xffffffffu, incl, n - 1);
        __syncwarp();
        published += total;
        /* No fence here: the published count only tells the service warps how many tickets they may
         * reserve; a ticket is taken when its own 16-byte word shows up (tag), whichever arrives first. */
        if (lane == 0 && total) *reinterpret_cast<volatile unsigned long long *>(g_published) = published;
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
    CtaCtl *c = reinterpret_cast<CtaCtl *>(smem + (ctrl - sbase));

#ifdef AESOFF_DEBUG
#define DBG_MIN(i) do { if (tid == 0 || (tid & 31u) == 0) atomicMin(reinterpret_cast<unsigned long long *>(P.counters) + 20 + (i), globaltimer_ns()); } while (0)
#define DBG_MAX(i) do { if (tid == 0 || (tid & 31u) == 0) atomicMax(reinterpret_cast<unsigned long long *>(P.counters) + 20 + (i), globaltimer_ns()); } while (0)
#else
#define DBG_MIN(i) ((void)0)
#define DBG_MAX(i) ((void)0)
#endif
    DBG_MIN(0); /* first CTA starts */
    DBG_MAX(1); /* last CTA starts  */
    /* Start-up: the worker warps build the tables (named barrier 2 among themselves) while the service
     * warp clears the control block and already fetches the first tickets; barrier 1 joins the two.  */
    const uint32_t warp = tid >> 5, lane = tid & 31u;
    if (warp == AESOFF_WORKER_WARPS) {
        for (uint32_t i = lane; i < CTRL_BYTES / 4; i += 32u) reinterpret_cast<uint32_t *>(c)[i] = 0u;
        __threadfence_block();
        asm volatile("bar.arrive 1, %0;" ::"n"(AESOFF_CTA_THREADS) : "memory");
        service_loop(P, c, lane);
    } else if (warp == AESOFF_WORKER_WARPS + 1) {
        asm volatile("bar.sync 1, %0;" ::"n"(AESOFF_CTA_THREADS) : "memory");
        if (P.mode == AESOFF_MODE_PERSISTENT && blockIdx.x == 0) dispatcher_loop(P, c, tbase | (lane * 4u), lane);
    } else {
        if (tid == 0 && blockIdx.x == 0 && P.hctl) P.hctl[AESOFF_CTL_SMEMBASE] = sbase;
        fill_tables(tbase, P.T0, tid, AESOFF_WORKER_WARPS * 32u); /* worker threads only */
        DBG_MAX(2); /* last CTA has its tables */
        asm volatile("bar.sync 1, %0;" ::"n"(AESOFF_CTA_THREADS) : "memory");
        worker_loop(P, c, tbase | (lane * 4u), lane);
        DBG_MIN(6); /* first worker warp leaves */
        DBG_MAX(7); /* last worker warp leaves  */
    }
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

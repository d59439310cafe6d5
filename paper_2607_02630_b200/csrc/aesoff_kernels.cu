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
 *   warp 17       DISPATCHER (CTAs 0 .. n_dispatchers-1, persistent mode only).  Polls the host-mapped
 *                 descriptor ring over PCIe (one round trip per batch of up to 32 requests; batches go
 *                 round the dispatcher warps), expands keys that arrive raw (step a1), and cuts each
 *                 request into chunk tickets (step a3).
 * Completion (step a7): the worker that finishes the last unit of a slot counts the request's chunks
 * down in global memory; the last chunk's finisher fences at system scope and writes the request's
 * sequence number into the host-mapped mailbox.
 */
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include <mutex>

#include "aesoff.h"
#include "aesoff_cipher.cuh"
#include "aesoff_internal.h"
#include "aesoff_shared.h"

using namespace aesoff;

namespace {

constexpr uint32_t AESOFF_STAGE_STRIDE = 36;
constexpr uint32_t AESOFF_LANDINGS = 4;      /* landing areas for polls of the host ring: up to three in flight + the one looked at */ /* words per staged descriptor: 32 + padding against bank conflicts */

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
    uint32_t mode;          /* AESOFF_MODE_CTR / _ECB_ENC / _ECB_DEC / _CBC_DEC                 */
    uint32_t pad_[2];
    uint32_t pad2_;         /* (the unit size lives in CtaCtl::unit_mode)                       */
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
    /* unit size of the slot's chunk: 0 rows (AESOFF_ROWS_PER_UNIT of them), AESOFF_FLAG_HALF, AESOFF_FLAG_FINE.  An array of
     * its own because the service warp reads it lane by lane for what the CTA holds: as a field of Slot (384 bytes apart,
     * i.e. one bank) that one load was a 16-way bank conflict and 1.2 % of the SM's shared-memory wavefronts (ncu, source page). */
    uint32_t unit_mode[AESOFF_SLOTS];
    uint32_t exit_flag;
    uint32_t disp_stat[4];        /* dispatcher: requests cut into 1/8 rows / half rows / rows so far, and "changed" */
    uint32_t tables_ready;        /* set by a worker once the tables are filled: the service warp, which starts fetching
                                     tickets while they are being built, needs them for a decrypting request's keys */
    uint32_t token_moved_us;      /* dispatcher: when it last saw the token move (1.024 us units; kept here, not in a register) */
    /* A dispatcher's CTA stands aside while requests overlap AND the GPU has nothing queued (service_loop): */
    uint32_t multi_until_us;      /* dispatcher: requests have been overlapping until about this time (1.024 us units)         */
    uint32_t last_take_us;        /* dispatcher: when it last took requests                                                    */
    uint32_t starved_us;          /* service warp: when it last found no ticket waiting                                        */
    uint32_t pad[2];
    /* dispatcher CTAs: landing areas for polls of the host ring (one is looked at while the next ones fly):
     * 32 descriptors as read from the ring, and a 33rd row for the control words that come with them */
    uint32_t stage[AESOFF_LANDINGS][33][AESOFF_STAGE_STRIDE];
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
__device__ __forceinline__ uint4 ld_volatile_v4(const void *p)
{
    uint4 v;
    asm volatile("ld.volatile.global.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "l"(p)
                 : "memory");
    return v;
}
/* 16 bytes global (or host-mapped) memory -> shared memory without a register in between: a poll in flight
 * holds no destination registers and no scoreboard that an LDS or SHFL of the code running under it could
 * end up waiting on (L2 only: mapped host memory is not cached on the GPU, every copy goes to the host) */
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gsrc)
                 : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
/* waits until at most `pending` of this thread's newest copy groups are still in flight (groups complete in order) */
__device__ __forceinline__ void cp_async_wait_but(uint32_t pending)
{
    if (pending == 0u)
        asm volatile("cp.async.wait_group 0;" ::: "memory");
    else if (pending == 1u)
        asm volatile("cp.async.wait_group 1;" ::: "memory");
    else
        asm volatile("cp.async.wait_group 2;" ::: "memory");
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
template <class PP>
__device__ __forceinline__ void complete_chunk(const PP &P, CtaCtl *c, uint32_t s)
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

/* NOT inlined into the kernel, and handed only the four pointers it needs: ptxas then allocates and schedules the
 * cipher loops by themselves.  Inlined beside the dispatcher and the service warp, the same source ran 0.6-0.9 % slower
 * after every change to THOSE roles (same instruction counts in the round loops, different schedule; found by timing the
 * drain-mode kernel of successive commits): 922 -> 934 GB/s at 1 MiB x 64, 652 -> 659 at AES-256 8 MiB x 16.        */
struct WorkerParams {
    uint32_t *dq_done;
    volatile uint64_t *hmail;
    uint64_t *dev_done_seq;
    uint64_t *counters;
};
__device__ __noinline__ void worker_loop(const WorkerParams P, CtaCtl *c, uint32_t ybase, uint32_t lane)
{
#ifdef AESOFF_DEBUG
    bool first = true;
#endif
#ifdef AESOFF_WSTATS
    /* -DAESOFF_WSTATS builds: per worker warp, clocks inside units and clocks between two units (waiting for work), so that
     * the persistent engine's own occupancy is measured, not extrapolated from a launch (aesoff_debug_worker_stats) */
    long long ws_busy = 0, ws_wait = 0, ws_prev = 0;
    unsigned long long ws_units = 0;
#endif
    for (;;) {
        const uint32_t got = claim_unit(c, lane);
#ifdef AESOFF_WSTATS
        const long long ws_t1 = clock64();
        if (got == CLAIM_EXIT) {
            if (lane == 0) {
                atomicAdd(reinterpret_cast<unsigned long long *>(P.counters) + AESOFF_CNT_DEBUG + 0, (unsigned long long)ws_busy);
                atomicAdd(reinterpret_cast<unsigned long long *>(P.counters) + AESOFF_CNT_DEBUG + 1, (unsigned long long)ws_wait);
                atomicAdd(reinterpret_cast<unsigned long long *>(P.counters) + AESOFF_CNT_DEBUG + 2, ws_units);
            }
            break;
        }
        if (ws_units) ws_wait += ws_t1 - ws_prev;
#endif
        if (got == CLAIM_EXIT) break;
#ifdef AESOFF_DEBUG
        if (lane == 0 && first) {
            atomicMin(reinterpret_cast<unsigned long long *>(P.counters) + AESOFF_CNT_DEBUG + 3, globaltimer_ns()); /* first unit claimed anywhere */
            atomicMax(reinterpret_cast<unsigned long long *>(P.counters) + AESOFF_CNT_DEBUG + 4, globaltimer_ns()); /* last warp gets its first unit */
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
        const uint32_t fine = c->unit_mode[s];
        if (sl->mode != AESOFF_MODE_CTR) {
            /* ECB / CBC-decrypt: the same units over rows of 256 blocks, no counter (the ICB words hold the IV) */
            const uint4 iv = make_uint4(sl->desc.icb[0], sl->desc.icb[1], sl->desc.icb[2], sl->desc.icb[3]);
            const uint32_t ybd = (ybase & ~0xffffu) + TD_OFF + (lane * 4u);
            uint64_t m = sl->unit0_row;
            uint32_t cnt = 1, kb0 = 0, kb1 = 8;
            if (fine & AESOFF_FLAG_FINE) {
                m += u >> 3;
                kb0 = u & 7u;
                kb1 = kb0 + 1u;
            } else if (fine & AESOFF_FLAG_HALF) {
                m += u >> 1;
                kb0 = (u & 1u) * 4u;
                kb1 = kb0 + 4u;
            } else {
                const uint32_t first = u * AESOFF_ROWS_PER_UNIT;
                m += first;
                cnt = sl->n_rows - first < AESOFF_ROWS_PER_UNIT ? sl->n_rows - first : AESOFF_ROWS_PER_UNIT;
            }
            if (kb1 - kb0 == 1u)
                mode_request_rows<1>(sl->mode, ybase, ybd, rk4, nr, iv, src, dst, len, m, cnt, lane, kb0, kb1);
            else
                mode_request_rows<4>(sl->mode, ybase, ybd, rk4, nr, iv, src, dst, len, m, cnt, lane, kb0, kb1);
        } else if (fine & AESOFF_FLAG_FINE) {
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
#ifdef AESOFF_WSTATS
        ws_prev = clock64();
        ws_busy += ws_prev - ws_t1;
        ++ws_units;
#endif
    }
}

/* ------------------------------------------------------------------------------------------ */
/* service warp: global ticket queue -> this CTA's slots, ahead of the workers  (a3)           */
/* ------------------------------------------------------------------------------------------ */
/* Lane j < AESOFF_SLOTS owns slot j.  All lanes run in lock step; nothing here is on the
 * workers' critical path as long as at least one slot is open.                                 */
__device__ void service_loop(const aesoff_params_t &P, CtaCtl *c, uint32_t ybase, uint32_t lane)
{
    unsigned long long *g_ticket = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_TICKET);
    const bool persistent = (P.mode == AESOFF_MODE_PERSISTENT);
    const bool mine = lane < AESOFF_SLOTS;
    unsigned long long *g_idle = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_IDLE);
    bool have = false;          /* this lane holds a reserved ticket for its (free) slot */
    unsigned long long t = 0;   /* that ticket */
    uint32_t stamp_base = 0;
    bool counted_idle = false;  /* this CTA is included in the device-wide idle-CTA count */
    uint32_t my_mode = 0;       /* unit size of the chunk in this lane's slot */
    /* a dispatcher warp runs beside this CTA's workers.  Such a CTA may stand aside (below) only while CTAs without a
     * dispatcher remain to take the tickets: in a grid of at most n_disp CTAs (n_ctas = 1 or 2 is allowed) nobody stands aside */
    const bool disp_cta = persistent && blockIdx.x < P.n_disp && gridDim.x > P.n_disp;
    uint32_t last_chunk_rows = P.chunk_rows; /* rows of the chunk this CTA read last (requests choose their chunk size) */

    for (;;) {
        /* this lane's slot: busy word and claim word, read together and ahead of the two L2 reads below (the claim word is
         * needed only after them, for what the CTA holds: read there, its shared-memory latency -- long while the workers
         * keep the pipe full -- came on top of the L2 round trip in every iteration) */
        uint32_t busy_w = 0, claim_w = 0;
        if (mine) {
            busy_w = lds_volatile(&c->busy[lane]);
            claim_w = lds_volatile(&c->claim[lane]);
        }
        const bool is_free = mine && busy_w == 0u;
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
        /* The CTA of a dispatcher warp stands aside -- reserves nothing -- while requests overlap (its dispatcher says so)
         * AND the queue has run dry within the last 24 us: then the GPU is short of work, not of CTAs, and what 16 cipher
         * warps cost the dispatcher beside them (issue slots on its sub-partition, the queue in front of the shared-memory
         * pipe that its loads and ticket stores go through too) is latency of every request.  With a lone request the
         * dispatcher has nothing to do while the request is worked on, and with a queue that never runs dry its speed
         * does not matter: in both cases the CTA works like any other.
         * (Measured with the two CTAs standing aside always: 1 MiB x 16 737 -> 773 GB/s, the mix 9.2 -> 9.9 M requests/s,
         * 64 KiB x 256 649 -> 664 GB/s -- and 938 -> 925 at saturation, which is why it is conditional.)              */
        bool stand_aside = false;
        if (disp_cta) {
            const uint32_t now = (uint32_t)(globaltimer_ns() >> 10);
            uint32_t starved = 0, until = 0;
            if (lane == 0) {
                if (avail == 0ull) sts_volatile(&c->starved_us, now);
                starved = avail == 0ull ? now : lds_volatile(&c->starved_us);
                until = lds_volatile(&c->multi_until_us);
            }
            stand_aside = __shfl_sync(0xffffffffu, (int)(until - now) > 0 && now - starved < 24u ? 1 : 0, 0) != 0;
        }
        /*    A CTA does not hoard: what it holds (unclaimed units of its open slots plus the tickets
         *    it has reserved, in 1/8-row units) stays near one and a half rows per worker -- enough
         *    to hide a refill (microseconds against 10 us per row), little enough that the end of a
         *    burst is not left to the few CTAs that grabbed 16 chunks each.                        */
        {
            const uint32_t per_ticket = last_chunk_rows * 8u; /* a reserved ticket that has not been read yet: as large as the last one */
            uint32_t held = 0;
            if (mine && !is_free) {
                const uint32_t w = claim_w;
                const uint32_t left = (w >> 16) > (w & 0xffffu) ? (w >> 16) - (w & 0xffffu) : 0u;
                const uint32_t f = my_mode; /* this lane filled the slot: it knows the unit size (CtaCtl::unit_mode is for the workers) */
                held = (f & AESOFF_FLAG_FINE) ? left : (f & AESOFF_FLAG_HALF) ? left * 4u : left * 8u * AESOFF_ROWS_PER_UNIT;
            } else if (have) {
                held = per_ticket;
            }
            held = __reduce_add_sync(0xffffffffu, held);
            /* The reservation on a ticket that does not exist yet: an idle CTA keeps one, and so does a CTA whose workers
             * are nearly out of work (less than half a row each): the ticket is then picked up one L2 round trip after it
             * is written instead of three (see the count, reserve, poll), which is latency that a window of small requests
             * turns into throughput.                                                                                  */
            if (persistent && !stand_aside && avail == 0ull && have_mask == 0u && (busy_mask == 0u || held < AESOFF_WORKER_WARPS * P.tune[AESOFF_TUNE_PRERESERVE]))
                avail = 1ull;
            const uint32_t hold_max = AESOFF_WORKER_WARPS * 12u; /* 1.5 rows per worker */
            unsigned long long cap = held < hold_max ? (hold_max - held + per_ticket - 1u) / per_ticket : 0u;
            if (cap == 0ull && busy_mask == 0u && have_mask == 0u) cap = 1ull;
            /* ... nor takes more than its share of a short queue: the last tickets of a burst (and the
             * tickets of a lone request) spread over all CTAs instead of piling up on the first few  */
            const uint32_t a32 = avail > 0x100000ull ? 0x100000u : (uint32_t)avail; /* 32-bit division */
            const uint32_t share = (a32 + gridDim.x - 1u) / gridDim.x;
            if (cap > share) cap = share ? share : 1ull;
            if (avail > cap) avail = cap;
            if (stand_aside) avail = 0ull;
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
            /* a decrypting request (ECB, CBC) runs the equivalent inverse cipher: its middle round keys go through
             * InvMixColumns, here, once per chunk (60 words, two per lane; 0.3 % of a 4-row chunk's lookups) */
            for (uint32_t m = ready_mask; m; m &= m - 1u) {
                const uint32_t sj = __ffs(m) - 1;
                Slot *sl = &c->slot[sj];
                const uint32_t md = sl->desc.flags & 3u;
                if (md == AESOFF_MODE_ECB_DEC || md == AESOFF_MODE_CBC_DEC) {
                    while (lds_volatile(&c->tables_ready) == 0u) __nanosleep(100);
                    uint32_t *rkw = reinterpret_cast<uint32_t *>(sl->rk4);
                    const uint32_t nrr = sl->desc.nr, ybd = (ybase & ~0xffffu) + TD_OFF + (lane * 4u);
                    for (uint32_t i = 4u + lane; i < 4u * nrr; i += 32u) rkw[i] = inv_mix_word(rkw[i], ybase, ybd);
                }
            }
            __syncwarp();
            uint32_t seen_rows = 0;
            if (ready) {
                Slot *sl = &c->slot[lane];
                const unsigned long long rows = sl->desc.rows;
                const uint32_t crows = sl->desc.chunk_rows;
                seen_rows = crows;
                const unsigned long long row0 = (unsigned long long)chunk * crows;
                const uint32_t nrows = (uint32_t)((rows - row0) < crows ? (rows - row0) : crows);
                const uint32_t fine = unit_mode & (AESOFF_FLAG_FINE | AESOFF_FLAG_HALF);
                const uint32_t n_units = (fine & AESOFF_FLAG_FINE) ? nrows * 8u : (fine & AESOFF_FLAG_HALF) ? nrows * 2u
                                         : (nrows + AESOFF_ROWS_PER_UNIT - 1u) / AESOFF_ROWS_PER_UNIT;
                sl->n_rows = nrows;
                sl->unit0_row = (uint32_t)row0;
                sl->ring_slot = ring;
                sl->n_units = n_units;
                c->unit_mode[lane] = fine;
                my_mode = fine;
                sl->mode = sl->desc.flags & 3u;
                c->done[lane] = 0u;
                c->stamp[lane] = stamp_base + __popc(ready_mask & ((1u << lane) - 1u));
                c->busy[lane] = 1u;
                __threadfence_block();
                sts_volatile(&c->claim[lane], n_units << 16); /* open the slot */
                have = false;
            }
            stamp_base += __popc(ready_mask);
            last_chunk_rows = __reduce_max_sync(0xffffffffu, seen_rows); /* ready_mask != 0: at least one lane saw one */
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
/* dispatcher warps (persistent mode, warp 17 of CTAs 0 .. n_disp-1): host ring -> tickets (a3) */
/* ------------------------------------------------------------------------------------------ */
/* Sequence numbers are dealt out in batches of 32: batch b = [first_seq + 32 b, +32) belongs to dispatcher
 * b % n_disp, lane k of that warp to request k of the batch.  A dispatcher reads its batch's ring slots
 * (8 when quiet, all 32 when busy; 128 B each, as 16-byte pieces that validate themselves, so there is no
 * flag-then-body dependency) in ONE PCIe round trip, and takes the ready prefix.
 *
 * Tickets are numbered in sequence order, so the dispatchers pass a token along: one 16-byte word
 * {tickets published, next sequence number to dispatch} in device memory (AESOFF_CNT_CHAIN).  A dispatcher
 * whose next request is chain.next holds the token: it sizes units and chunks by the load it sees, adds
 * its ticket count, stores the word for the next one -- a fraction of a microsecond -- and only then does
 * the long part (key expansion for raw keys, descriptors, tickets) beside the other dispatchers.  The word
 * is read with every poll, so a lone request never waits for it.                                         */
__device__ void dispatcher_loop(const aesoff_params_t &P, CtaCtl *c, uint32_t ybase, uint32_t lane, uint32_t d)
{
    unsigned long long *g_published = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_PUBLISHED);
    unsigned long long *g_stop = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_STOP);
    unsigned long long *g_quit = reinterpret_cast<unsigned long long *>(P.counters + AESOFF_CNT_QUIT);
    uint4 *g_chain = reinterpret_cast<uint4 *>(P.counters + AESOFF_CNT_CHAIN);
    const uint32_t Rm = P.R - 1;
    const uint32_t K = P.n_disp;
    unsigned long long b_seq = P.first_seq + (unsigned long long)AESOFF_BATCH * d; /* first request of my batch   */
    uint32_t pos = 0;                          /* requests of it already dispatched            */
    bool have_token = false;                   /* chain.next == b_seq + pos, and I know it     */
    unsigned long long my_pub = 0;             /* chain.published while I hold the token       */
    unsigned long long oldest = P.first_seq;   /* every seq below this is known to be complete */
    unsigned long long base = 0;               /* first ticket of request `oldest` at the last scan */
    uint32_t last_activity_us = (uint32_t)(globaltimer_ns() >> 10), seen_next = 0; /* dispatcher 0's idle timer (1.024 us units) */
    uint32_t wide = 0;                         /* 0: poll 8 slots, 1: poll 32                  */
#ifdef AESOFF_DISP_STATS
    uint32_t dbg_takes = 0, dbg_reqs = 0, dbg_empty = 0;
    unsigned long long dbg_wait = 0, dbg_work = 0;
#endif

    if (lane == 0 && d == 0) P.hctl[AESOFF_CTL_ALIVE] = 1;

    /* One poll = ring slots of my batch as 16-byte pieces (piece g = 32 j + lane: slot q + g / 8 of the batch,
     * piece g % 8), plus the host's control words and three device words: the token, {tickets reserved, published}
     * and {idle CTAs, quit}.  All of it is copied asynchronously (cp.async) into the landing area the warp is NOT
     * looking at, and a poll is issued as soon as the previous one has been looked at, i.e. BEFORE that batch is
     * processed: the PCIe round trip of the next one runs under the on-chip work of this one.  (The polls used to
     * live in 32 registers; whenever ptxas let an LDS of the processing code share a scoreboard with them, that
     * LDS waited out the PCIe round trip: +1.6 us on every request, found with a time stamp.)                */
    uint32_t cur = 0;                      /* landing area being looked at */
    uint32_t n_issued = 0, n_looked = 0;   /* polls issued / looked at: area of poll i is i % AESOFF_LANDINGS */
#define AUX_CTL   0   /* row 32 of a landing area: words 0..3 host control words (0 = stop) */
#define AUX_CHAIN 4   /*   4..7   the token                                                  */
#define AUX_TKT   8   /*   8..11  {tickets reserved, tickets published}                      */
#define AUX_IDLE  12  /*   12..15 {idle CTAs, quit, long queue}                              */
#define ISSUE_POLL(bseq, q, ring)                                                                            \
    do {                                                                                                     \
        uint32_t(*land_)[AESOFF_STAGE_STRIDE] = c->stage[n_issued++ % AESOFF_LANDINGS];                      \
        const uint32_t nload_ = !(ring) ? 0u : wide ? 8u : 2u;                                               \
        const uint32_t q_ = wide ? 0u : (q);                                                                 \
        _Pragma("unroll") for (uint32_t j = 0; j < 8; ++j)                                                  \
        {                                                                                                    \
            const uint32_t k_ = q_ + j * 4u + (lane >> 3);                                                   \
            if (j < nload_ && k_ < AESOFF_BATCH) {                                                           \
                const uint32_t sl_ = (uint32_t)(((bseq) + k_ - 1) & Rm);                                     \
                cp_async16(&land_[k_][4u * (lane & 7u)], reinterpret_cast<const uint8_t *>(P.hring + sl_) + 16u * (lane & 7u)); \
            }                                                                                                \
        }                                                                                                    \
        if (lane == 0) {                                                                                     \
            if (ring)                                                                                        \
                cp_async16(&land_[32][AUX_CTL], const_cast<const uint32_t *>(P.hctl));                       \
            else                                                                                             \
                land_[32][AUX_CTL + AESOFF_CTL_STOP] = 0u;                                                   \
        } else if (lane < 4) {                                                                               \
            cp_async16(&land_[32][4u * lane], P.counters + (lane == 1 ? AESOFF_CNT_CHAIN : lane == 2 ? AESOFF_CNT_TICKET : AESOFF_CNT_IDLE)); \
        }                                                                                                    \
        cp_async_commit();                                                                                   \
    } while (0)
    /* Only the dispatcher that holds the token can take requests now; what the others read is a prefetch.  Polls
     * of several warps queue up behind one another on PCIe (four of them polling flat out added 4 us to a lone
     * request), so: the holder polls continuously; the others only watch the token -- unless the holder has
     * found a long queue (eight or more requests ready at once: it says so in a device word), in which case
     * the dispatchers whose batch comes next or next but one read their slots ahead of the token.            */
    unsigned long long token_at = (K == 1u) ? b_seq : 0ull; /* chain.next as last seen */
    bool queue_long = false;     /* the holder's last word on it */
    uint32_t empties = 0;        /* looks in a row that found nothing */
    if (lane == 0) c->token_moved_us = (uint32_t)(globaltimer_ns() >> 10) - 1000u;
    __syncwarp();

    for (;;) {
        /* ---- phase 1: the PCIe round trip ---------------------------------------------------- */
        {
            const bool holder = have_token || token_at == b_seq + pos;
            /* ... and the warp whose batch comes next reads its slots ahead once the holder has at most four requests
             * of its batch left and the token has moved in the last few microseconds (traffic, not an idle engine whose
             * token happens to rest there): without this, every 32nd request of a moderate stream waited for the next
             * warp to wake up (3 us) and for its first poll (1.5 us) -- 1 MiB x 16: 729 -> 741 GB/s, p99 31.8 -> 29.1 us                    */
            const uint32_t now_us = (uint32_t)(globaltimer_ns() >> 10);
            const bool soon = !holder && b_seq + pos <= token_at + 4ull && now_us - lds_volatile(&c->token_moved_us) < 8u;
            const bool near = holder || soon || (queue_long && token_at + 2ull * AESOFF_BATCH >= b_seq);
            /* The holder of the token, once it has found the ring empty (an idle engine: the latency case), keeps `depth` polls in flight, each issued when an older one has been looked at: a request
             * that arrives waits a fraction of a PCIe round trip for the next poll to leave instead of half of one
             * (lone 4 KiB 8.9 -> 8.25 us with three; 3 KiB per microsecond of PCIe reads).  Polls that were issued before
             * a request was taken would show it again: they are skipped, not looked at (see the end of the loop).   */
            const uint32_t depth = (holder && empties >= 1u) ? P.tune[AESOFF_TUNE_POLL_DEPTH] : 1u;
            if (!holder && !soon && n_issued == n_looked) __nanosleep(queue_long ? 400u : 3000u); /* device words only: no PCIe read (ISSUE_POLL) */
            while (n_issued - n_looked < depth) {
                if (n_issued != n_looked) __nanosleep(P.tune[AESOFF_TUNE_POLL_GAP]); /* spread them over a round trip */
                ISSUE_POLL(b_seq, pos, near);
            }
        }
        cp_async_wait_but(n_issued - n_looked - 1u);
        cur = n_looked++ % AESOFF_LANDINGS;
        __syncwarp();
#ifdef AESOFF_DISP_STATS
        const unsigned long long dbg_t0 = globaltimer_ns(); /* the poll has landed */
#endif
        /* lane k looks at request k of the batch (rows outside this poll hold older pieces: their tags
         * either still match, from an earlier poll of this batch, or belong to another batch) */
        const unsigned long long s = b_seq + lane;
        const uint32_t slot = (uint32_t)((s - 1) & Rm);
        const uint32_t *sw = c->stage[cur][lane];
        const uint32_t *ax = c->stage[cur][32];
        const uint32_t tag = (uint32_t)s;
        /* the first line of the descriptor in four 16-byte reads, kept in registers for the whole take: under load the
         * dispatcher's shared-memory reads queue behind its SM's table lookups, so there are few of them
         * (pieces: {ICB0..2} {ICB3, src} {dst, len lo} {len hi, key word, mode}, each with its tag) */
        const uint4 p0 = *reinterpret_cast<const uint4 *>(sw + 0), p1 = *reinterpret_cast<const uint4 *>(sw + 4);
        const uint4 p2 = *reinterpret_cast<const uint4 *>(sw + 8), p3 = *reinterpret_cast<const uint4 *>(sw + 12);
        const uint32_t kw = p3.y;
        bool valid = lane >= pos && p0.w == tag && p1.w == tag && p2.w == tag && p3.w == tag;
        if (valid && (kw & AESOFF_KW_RAW)) valid = sw[19] == tag && sw[23] == tag && sw[27] == tag && sw[31] == tag;
        const uint32_t vrun = ~(__ballot_sync(0xffffffffu, valid) >> pos); /* bit i: request pos + i is not ready */
        uint32_t n = vrun ? (uint32_t)(__ffs(vrun) - 1) : 32u;           /* length of the ready run from pos */
        if (n > 32u - pos) n = 32u - pos;
        const uint4 a_ctl = *reinterpret_cast<const uint4 *>(ax + AUX_CTL), a_chain = *reinterpret_cast<const uint4 *>(ax + AUX_CHAIN);
        const uint4 a_tkt = *reinterpret_cast<const uint4 *>(ax + AUX_TKT), a_idle = *reinterpret_cast<const uint4 *>(ax + AUX_IDLE);
        const uint32_t stop = a_ctl.x; /* AESOFF_CTL_STOP is word 0 */
        unsigned long long chain_pub = ((unsigned long long)a_chain.y << 32) | a_chain.x;
        unsigned long long chain_next = ((unsigned long long)a_chain.w << 32) | a_chain.z;
        const unsigned long long reserved = ((unsigned long long)a_tkt.y << 32) | a_tkt.x;
        const unsigned long long idle = ((unsigned long long)a_idle.y << 32) | a_idle.x;
        const uint32_t quit_word = a_idle.z;
        queue_long = a_idle.w != 0u;
        if (chain_next != token_at && lane == 0) {
            /* another dispatcher has taken requests: the same bookkeeping as for a take of this warp's own (below) */
            const uint32_t now = (uint32_t)(globaltimer_ns() >> 10);
            sts_volatile(&c->token_moved_us, now);
            if (chain_next - token_at >= 2ull || now - c->last_take_us < 7u) sts_volatile(&c->multi_until_us, now + 32u);
            c->last_take_us = now;
        }
        token_at = chain_next;
        wide = (n >= 8u) ? 1u : 0u;
        const uint32_t n_seen = n;
#ifdef AESOFF_EARLY_PREFETCH
        if (n != 0) { /* the next poll lands in the other area */
            if (pos + n == 32u)
                ISSUE_POLL(b_seq + (unsigned long long)AESOFF_BATCH * K, 0u, true);
            else
                ISSUE_POLL(b_seq, pos + n, true);
        }
#endif
        empties = n ? 0u : empties + 1u;
        if (n == 0) {
            if (queue_long && (have_token || chain_next == b_seq + pos)) { /* the queue has run dry: the others stop reading ahead */
                queue_long = false;
                if (lane == 0) *(reinterpret_cast<volatile uint32_t *>(g_quit) + 1) = 0u;
            }
#ifdef AESOFF_DISP_STATS
            ++dbg_empty;
#endif
            if (c->disp_stat[3]) {
                /* not on a request's way: a PCIe write in flight would hold up the next fence */
                if (lane == 0) {
                    volatile uint32_t *st = P.hctl + AESOFF_CTL_STATS + AESOFF_CTL_STAT_WORDS * d;
                    st[AESOFF_CTL_CUT_EIGHTHS] = c->disp_stat[0];
                    st[AESOFF_CTL_CUT_HALVES] = c->disp_stat[1];
                    st[AESOFF_CTL_CUT_ROWS] = c->disp_stat[2];
                    c->disp_stat[3] = 0u;
#ifdef AESOFF_DISP_STATS
                    st[AESOFF_CTL_DBG_TAKES] = dbg_takes;
                    st[AESOFF_CTL_DBG_REQS] = dbg_reqs;
                    st[AESOFF_CTL_DBG_WAIT] = (uint32_t)(dbg_wait >> 6);
                    st[AESOFF_CTL_DBG_WORK] = (uint32_t)(dbg_work >> 6);
                    st[AESOFF_CTL_DBG_EMPTY] = dbg_empty;
#endif
                }
                __syncwarp();
            }
            bool quit = stop != 0 || quit_word != 0;
            if (!quit && d == 0 && P.idle_exit_ms) {
                /* the idle timer is dispatcher 0's: it runs while no dispatcher takes anything, and fires only
                 * when everything that was accepted has completed */
                const uint32_t now = (uint32_t)(globaltimer_ns() >> 10);
                if ((uint32_t)chain_next != seen_next) {
                    seen_next = (uint32_t)chain_next;
                    last_activity_us = now;
                } else if (now - last_activity_us > P.idle_exit_ms * 977u) {
                    if (chain_next > oldest + P.R) oldest = chain_next - P.R;
                    for (;;) {
                        const unsigned long long q = oldest + lane;
                        bool fin = false;
                        if (q < chain_next)
                            fin = *reinterpret_cast<volatile uint64_t *>(P.dev_done_seq + ((q - 1) & Rm)) >= q;
                        const uint32_t fm = __ballot_sync(0xffffffffu, fin);
                        const uint32_t adv = (fm == 0xffffffffu) ? 32u : (uint32_t)(__ffs(~fm) - 1);
                        oldest += adv;
                        if (adv < 32u) break;
                    }
                    if (oldest >= chain_next)
                        quit = true;
                    else
                        last_activity_us = now;
                }
            }
            if (quit) {
                /* the host stops the engine only after everything has completed, and only a dispatcher that reads
                 * the ring reads the host's stop word: the first to see it tells the others (quit word), lets the
                 * service warps go and reports the exit */
                if (lane == 0 && quit_word == 0u) {
                    *reinterpret_cast<volatile uint32_t *>(g_quit) = 1u;
                    st_release_gpu(g_stop, 1ull);
                    __threadfence_system();
                    P.hctl[AESOFF_CTL_ALIVE] = 2;
                }
                return;
            }
            continue;
        }

        /* ---- phase 2: what does not depend on the token: the rows of request pos + k ---------------- */
        /* (32-bit row counts: the host refuses requests of 2^36 bytes and more, check_buffers) */
        const bool mine = lane >= pos && lane < pos + n;
        uint32_t rows = 0;
#define PW(p) sw[AESOFF_PW_INDEX(p)]
        if (mine) {
            const unsigned long long len = ((unsigned long long)p3.x << 32) | p2.z;
            const unsigned long long nblocks = (len >> 4) + ((len & 15ull) ? 1ull : 0ull);
            const uint32_t c0 = (p3.z & 3u) ? 0u : p1.x >> 24; /* rows start at counter byte 0 (CTR) or at the payload's start */
            rows = nblocks ? (uint32_t)((nblocks + c0 + AESOFF_ROW_BLOCKS - 1) >> 8) : 0u;
        }
        /* rows of this poll up to and including request k */
        uint32_t rows_incl = rows;
        if (n > 1) { /* a lone request (the latency case) skips the scan */
#pragma unroll
            for (int dd = 1; dd < 32; dd <<= 1) {
                const uint32_t y = __shfl_up_sync(0xffffffffu, rows_incl, dd);
                if ((int)lane >= dd) rows_incl += y;
            }
        }
        const uint32_t rows_poll = __shfl_sync(0xffffffffu, rows_incl, n > 1 ? 31 : (int)pos);

        const unsigned long long my_next = b_seq + pos;
        /* the published count as this poll saw it (the reserved count and the idle CTAs come from the same poll): the
         * load figures are heuristics, and sizing the requests BEFORE the token arrives keeps the token's holding time
         * -- the one serial step of the dispatchers -- down to a sum, a ballot and a store */
        const unsigned long long pub_est = have_token ? my_pub : chain_pub;
        /* Unit and chunk sizes by the load the request meets (all in 4 KiB rows; W = worker warps of the grid):
         *   backlog   rows published and not yet reserved by any CTA (chunk_rows per ticket, roughly)
         *   ahead     backlog + the rows of the requests before it in this poll
         *   total     backlog + all rows of this poll: the queue as far as it is known
         *   idle GPU  a quarter of the CTAs or more have no open slot
         * Per chunk (the unit size travels in the ticket), r0 rows into its request:
         *   1/8 rows   idle GPU, and the whole known queue is short (tune[FINE_TOTAL]) or the chunk is among its
         *              first tune[FINE_FRONT] rows: spread it over every warp, nobody waits for the extra lookups
         *   half rows  the known queue is at most tune[HALF_TOTAL] rows, or the request found at most tune[TAIL_AHEAD]
         *              rows ahead of it and the chunk is among the last tune[TAIL_LEFT] rows of the queue (the end
         *              of a long lone request must not be left to the few warps holding 2-row units)
         *   rows       otherwise (saturation: 135.3 lookups per block instead of 139.75 / 160)
         * Chunk = what one CTA takes at a time.  An idle CTA waits on ONE ticket that does not exist yet, so a request
         * that finds (nearly) every CTA idle and at most tune[SPREAD_AHEAD] rows ahead is cut into one chunk per CTA,
         * if that makes chunks of at most tune[SPREAD_MAX] rows: every CTA gets its share in the first round of
         * ticket reads.  Otherwise a chunk is chunk_rows rows: small enough to balance, large enough that the
         * service warps keep up.                                                                             */
        uint32_t fine_max, half_min; /* the chunk that starts r0 rows into this lane's request: 1/8 rows if
                                        (int)r0 <= fine_max, else half rows if (int)r0 >= half_min, else rows */
        /* (the dispatcher is one warp running dependent instructions, a few clocks each: a hundred instructions
         * on this path are 0.2 us on every request, so chunk sizes are powers of two and nothing here divides) */
        uint32_t nchunks = 0, clog = P.chunk_log2; /* rows per chunk = 1 << clog ... */
        uint32_t spread_rows = 0;                  /* ... unless this says otherwise (a lone request: one chunk per CTA) */
        {
            const unsigned long long bl = (pub_est > reserved ? pub_est - reserved : 0ull) << P.chunk_log2;
            const uint32_t backlog = bl > 0x3fffffffull ? 0x3fffffffu : (uint32_t)bl;
            const uint32_t total_q = min(backlog + min(rows_poll, 0x3fffffffu), 0x3fffffffu);
            const uint32_t ahead = min(backlog + (rows_incl - rows), 0x3fffffffu);
            const bool may_cut = P.fine_rows != 0u && rows <= P.fine_rows;
            const bool idle_gpu = idle * 4ull >= (unsigned long long)gridDim.x;
            if (mine && may_cut && idle * 8ull >= 7ull * gridDim.x && ahead <= P.tune[AESOFF_TUNE_SPREAD_AHEAD] &&
                rows <= gridDim.x * P.tune[AESOFF_TUNE_SPREAD_MAX]) { /* a lone request of moderate size */
                /* longer requests keep chunk_rows: many tickets per CTA balance by themselves, and what a CTA may
                 * hold is counted in chunk_rows-sized tickets (service_loop) */
                /* (not a power of two: 8 MiB is 2,048 rows, and 128 chunks of 16 would leave 20 of 148 CTAs without any;
                 * the two divisions are paid by requests longer than one row per CTA only) */
                clog = 0;
                if (rows > gridDim.x) spread_rows = (rows + gridDim.x - 1u) / gridDim.x;
            } else if (mine && may_cut && rows >= 4u * gridDim.x * AESOFF_WORKER_WARPS) {
                /* a very long request (37 MiB and up): 16-row chunks, a quarter of the tickets -- cut into 4-row chunks a lone
                 * 64 MiB request ran at 747 GB/s, the service warps' ticket and descriptor traffic being what held it back;
                 * with 16-row chunks 789.  (What a CTA may hold is counted in rows of the chunks it has seen: service_loop.) */
                clog = max(clog, 4u);
            } else if (mine && may_cut && rows >= 64u && total_q >= 4u * gridDim.x * AESOFF_WORKER_WARPS) {
                clog = max(clog, 3u); /* saturation: 8-row chunks, half the slot fills (8 MiB x 16: 938 -> 942 GB/s, AES-256 661 -> 664) */
            }
            int fm = -1, hm = 0x7fffffff;
            if (may_cut) {
                if (idle_gpu)
                    fm = total_q <= P.tune[AESOFF_TUNE_FINE_TOTAL] ? 0x7fffffff
                                                                   : (int)P.tune[AESOFF_TUNE_FINE_FRONT] - (int)ahead - (int)(spread_rows ? spread_rows : 1u << clog);
                if (total_q <= P.tune[AESOFF_TUNE_HALF_TOTAL])
                    hm = 0;
                else if (ahead <= P.tune[AESOFF_TUNE_TAIL_AHEAD])
                    hm = max(0, (int)(total_q - ahead) - (int)P.tune[AESOFF_TUNE_TAIL_LEFT]);
            }
            fine_max = (uint32_t)fm;
            half_min = (uint32_t)hm;
        }
#define UNIT_MODE(fm_, hm_, r0_) ((int)(r0_) <= (int)(fm_) ? AESOFF_FLAG_FINE : (int)(r0_) >= (int)(hm_) ? AESOFF_FLAG_HALF : 0u)
        if (mine) {
            /* a request must fit the ticket ring with room to spare */
            while (((rows + (1u << clog) - 1u) >> clog) > P.TM / 4u) ++clog;
            nchunks = (rows + (1u << clog) - 1u) >> clog;
            if (spread_rows) nchunks = (rows + spread_rows - 1u) / spread_rows;
        }
        const uint32_t crows = spread_rows ? spread_rows : 1u << clog; /* rows per chunk of this lane's request */
        /* exclusive prefix sum of nchunks -> first ticket of each request */
        uint32_t incl = nchunks;
        if (n > 1) {
#pragma unroll
            for (int dd = 1; dd < 32; dd <<= 1) {
                const uint32_t y = __shfl_up_sync(0xffffffffu, incl, dd);
                if ((int)lane >= dd) incl += y;
            }
        }
        /* ---- phase 3: the token -------------------------------------------------------------------- */
        /* (everything above ran while it was on its way: what its holder still does is a sum, a ballot and a store) */
        if (have_token) {
            chain_pub = my_pub;
        } else {
            /* only the token is read again: the load figures of the poll are heuristics, and the line the
             * ticket counter lives on belongs to the service warps' atomics */
            while (chain_next != my_next) {
                uint4 v = make_uint4(0, 0, 0, 0);
                if (lane == 0) v = ld_volatile_v4(P.counters + AESOFF_CNT_CHAIN);
                chain_pub = ((unsigned long long)__shfl_sync(0xffffffffu, v.y, 0) << 32) | __shfl_sync(0xffffffffu, v.x, 0);
                chain_next = ((unsigned long long)__shfl_sync(0xffffffffu, v.w, 0) << 32) | __shfl_sync(0xffffffffu, v.z, 0);
            }
        }
        const unsigned long long published = chain_pub;
#ifdef AESOFF_DISP_STATS
        const unsigned long long dbg_t1 = globaltimer_ns();
        dbg_wait += dbg_t1 - dbg_t0;
        ++dbg_takes;
#endif
        const unsigned long long first_ticket = published + incl - nchunks;
        /* ticket-ring capacity: every unfinished ticket must stay within TM of the newest.  `base`
         * is only refreshed (32 completion words per L2 round trip) when the cached one says no. */
        for (;;) {
            const uint32_t fits = __ballot_sync(0xffffffffu, !mine || first_ticket + nchunks - base <= P.TM) >> pos;
            uint32_t nfit = (~fits) ? (uint32_t)(__ffs(~fits) - 1) : 32u;
            if (nfit >= n) break;
            /* a ring slot is reused only after its previous request completed: whatever is a ring's length behind
             * the request in hand needs no look (this bounds the scan after a long run without one) */
            if (my_next > oldest + P.R) oldest = my_next - P.R;
            for (;;) {
                const unsigned long long q = oldest + lane;
                bool fin = false;
                if (q < my_next) fin = *reinterpret_cast<volatile uint64_t *>(P.dev_done_seq + ((q - 1) & Rm)) >= q;
                const uint32_t fm = __ballot_sync(0xffffffffu, fin);
                const uint32_t adv = (fm == 0xffffffffu) ? 32u : (uint32_t)(__ffs(~fm) - 1);
                oldest += adv;
                if (adv < 32u) break;
            }
            /* first ticket of the oldest unfinished request: piece 6 of its device descriptor, which another
             * dispatcher may not have written yet (then the tag is an older one, and the bound stays) */
            unsigned long long nb = base;
            if (oldest >= my_next) {
                nb = published;
            } else if (lane == 0) {
                const uint4 v = ld_volatile_v4(&P.dq[(oldest - 1) & Rm].w[24]);
                if (v.w == (uint32_t)oldest) nb = ((unsigned long long)v.y << 32) | v.x;
            }
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
        const bool take = lane >= pos && lane < pos + n;
        if (!take) nchunks = 0;
        const uint32_t total = __shfl_sync(0xffffffffu, incl, pos + n - 1);
        /* pass the token on: everything below runs beside the other dispatchers */
        const unsigned long long new_pub = published + total;
        if (lane == 0) {
            const unsigned long long nx = my_next + n;
            asm volatile("st.volatile.global.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(g_chain), "r"((uint32_t)new_pub),
                         "r"((uint32_t)(new_pub >> 32)), "r"((uint32_t)nx), "r"((uint32_t)(nx >> 32))
                         : "memory");
        }
        if (K > 1u && (wide != 0u) != queue_long) { /* as the holder: tell the others whether reading ahead pays */
            queue_long = wide != 0u;
            if (lane == 0) *(reinterpret_cast<volatile uint32_t *>(g_quit) + 1) = wide;
        }
        have_token = pos + n < 32u || K == 1u; /* still mine: nobody else can move it */
        my_pub = new_pub;
        token_at = my_next + n;

        /* ---- phase 4: keys, descriptors, tickets ----------------------------------------------- */
        const uint32_t fine = UNIT_MODE(fine_max, half_min, 0u); /* of the request's first chunk (statistics, descriptor) */
        uint32_t keyloc = kw & 0xffffu;
        if (!(kw & AESOFF_KW_RAW) && keyloc >= AESOFF_KEY_IDS) keyloc = AESOFF_KEY_IDS + slot; /* never sent by the host */
        if (take && (kw & AESOFF_KW_RAW)) {
            if (!(kw & AESOFF_KW_INSTALL) || keyloc >= AESOFF_KEY_IDS) keyloc = AESOFF_KEY_IDS + slot;
            uint32_t key[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) key[i] = PW(AESOFF_PW_RAWKEY + i);
            const uint32_t nr = kw >> 24;
            if (nr == 10)
                key_expand<4>(ybase, key, P.ktab[keyloc].rk); /* step a1 on the device */
            else if (nr == 12)
                key_expand<6>(ybase, key, P.ktab[keyloc].rk);
            else
                key_expand<8>(ybase, key, P.ktab[keyloc].rk);
        }
#undef PW
        /* expanded keys (if any request of this poll brought a raw one) before the tickets that point at
         * them; descriptors need no fence, their pieces validate themselves */
        if (__any_sync(0xffffffffu, take && (kw & AESOFF_KW_RAW))) __threadfence();
        __syncwarp();
        /* a request of up to eight chunks (the fine-grained regime: every request of the poll) gets its
         * tickets from its own lane; the warp then shares out the long ones, 32 tickets per step (all of their
         * tickets: the per-lane loop costs the warp as many passes as its longest request has chunks) */
        if (take && nchunks <= 8u) {
            for (uint32_t ch = 0; ch < nchunks; ++ch) {
                const unsigned long long tno = first_ticket + ch;
                const uint32_t md = UNIT_MODE(fine_max, half_min, ch * crows) << AESOFF_TICKET_MODE_SHIFT;
                *reinterpret_cast<uint4 *>(P.tmap + (tno & (unsigned long long)(P.TM - 1))) =
                    make_uint4((uint32_t)s, ch | md, keyloc, (uint32_t)tno + 1u);
            }
        }
        for (uint32_t big = __ballot_sync(0xffffffffu, take && nchunks > 8u); big; big &= big - 1u) {
            const uint32_t k = __ffs(big) - 1;
            const uint32_t nc = __shfl_sync(0xffffffffu, nchunks, k);
            const unsigned long long ft = __shfl_sync(0xffffffffu, first_ticket, k);
            const uint32_t kl = __shfl_sync(0xffffffffu, keyloc, k);
            const uint32_t cl = __shfl_sync(0xffffffffu, crows, k);
            const uint32_t fm = __shfl_sync(0xffffffffu, fine_max, k), hm = __shfl_sync(0xffffffffu, half_min, k);
            const uint32_t sq = (uint32_t)(b_seq + k);
            for (uint32_t ch = lane; ch < nc; ch += 32) {
                const unsigned long long tno = ft + ch;
                const uint32_t md = UNIT_MODE(fm, hm, ch * cl) << AESOFF_TICKET_MODE_SHIFT;
                *reinterpret_cast<uint4 *>(P.tmap + (tno & (unsigned long long)(P.TM - 1))) =
                    make_uint4(sq, ch | md, kl, (uint32_t)tno + 1u);
            }
        }
#undef UNIT_MODE
        /* the descriptors AFTER the tickets: a service warp that waits on a ticket reads it one L2 round trip after it
         * is written and only then asks for the descriptor, whose pieces validate themselves (a piece read too early
         * is read again); the eight stores per request used to stand between a request and its first ticket */
        if (take) {
            /* the 24 descriptor words as 8 pieces of {3 words, tag}: see aesoff_dq_entry_t */
            uint4 *d4 = reinterpret_cast<uint4 *>(P.dq + slot);
            const uint32_t tg = (uint32_t)s;
            d4[0] = p0; /* the first three pieces as they came (their tag is this request's) */
            d4[1] = p1;
            d4[2] = p2;
            d4[3] = make_uint4(p3.x, kw >> 24, p3.z & 3u, tg);
            d4[4] = make_uint4(nchunks, crows, (uint32_t)s, tg);
            d4[5] = make_uint4((uint32_t)(s >> 32), rows, 0u, tg);
            d4[6] = make_uint4((uint32_t)first_ticket, (uint32_t)(first_ticket >> 32), keyloc, tg);
            d4[7] = make_uint4(0u, 0u, 0u, tg);
        }
        __syncwarp();
        /* What the service warps read, raised once the tickets are on their way.  Not a store: a dispatcher that got
         * the token later may already have published a larger count.  No fence: the count only tells the service warps
         * how many tickets they may reserve; a ticket is taken when its own 16-byte word shows up (tag).          */
        if (lane == 0 && total) atomicMax(g_published, new_pub);
        if (lane == 0) { /* do requests overlap?  Two or more in one take, or two takes within 7 us (a lone request takes 8.7) */
            const uint32_t now = (uint32_t)(globaltimer_ns() >> 10);
            if (n >= 2u || now - c->last_take_us < 7u) sts_volatile(&c->multi_until_us, now + 32u);
            c->last_take_us = now;
        }
        {   /* statistics for aes_engine_info */
            const uint32_t me = __ballot_sync(0xffffffffu, take && (fine & AESOFF_FLAG_FINE));
            const uint32_t mh = __ballot_sync(0xffffffffu, take && (fine & AESOFF_FLAG_HALF));
            if (lane == 0) { /* kept in shared memory, not in registers; written to the host when the ring is next found empty */
                c->disp_stat[0] += __popc(me);
                c->disp_stat[1] += __popc(mh);
                c->disp_stat[2] += n - __popc(me) - __popc(mh);
                c->disp_stat[3] = 1u;
            }
        }
        /* an empty request (len == 0) has no ticket: complete it here */
        if (take && nchunks == 0) {
            __threadfence_system();
            P.hmail[slot] = s;
            *reinterpret_cast<volatile uint64_t *>(P.dev_done_seq + slot) = s;
        }
#ifdef AESOFF_DISP_STATS
        dbg_reqs += n;
        dbg_work += globaltimer_ns() - dbg_t1;
#endif
#ifndef AESOFF_EARLY_PREFETCH
        /* the next poll, after the last ticket store: issuing the copies takes a quarter of a microsecond that a lone
         * request would otherwise wait for; under load the poll still flies while the service warps pick the
         * tickets up and while this warp does the look and the token of the next batch */
        if (n == n_seen) {
            if (pos + n == 32u)
                ISSUE_POLL(b_seq + (unsigned long long)AESOFF_BATCH * K, 0u, true);
            else
                ISSUE_POLL(b_seq, pos + n, true);
            n_looked = n_issued - 1u; /* older polls in flight are stale: wait them out with this one, do not look */
        } else {
            n_looked = n_issued;
        }
#endif
        pos += n;
        if (pos == 32u) {
            pos = 0;
            b_seq += (unsigned long long)AESOFF_BATCH * K;
        }
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
    const uint32_t ctrl = (tbase - sbase >= CTRL_BYTES) ? sbase : tbase + TABLE_BYTES + TD_BYTES;
    CtaCtl *c = reinterpret_cast<CtaCtl *>(smem + (ctrl - sbase));

#ifdef AESOFF_DEBUG
#define DBG_MIN(i) do { if (tid == 0 || (tid & 31u) == 0) atomicMin(reinterpret_cast<unsigned long long *>(P.counters) + AESOFF_CNT_DEBUG + (i), globaltimer_ns()); } while (0)
#define DBG_MAX(i) do { if (tid == 0 || (tid & 31u) == 0) atomicMax(reinterpret_cast<unsigned long long *>(P.counters) + AESOFF_CNT_DEBUG + (i), globaltimer_ns()); } while (0)
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
        service_loop(P, c, tbase | (lane * 4u), lane);
    } else if (warp == AESOFF_WORKER_WARPS + 1) {
        asm volatile("bar.sync 1, %0;" ::"n"(AESOFF_CTA_THREADS) : "memory");
        if (P.mode == AESOFF_MODE_PERSISTENT && blockIdx.x < P.n_disp) dispatcher_loop(P, c, tbase | (lane * 4u), lane, blockIdx.x);
    } else {
        if (tid == 0 && blockIdx.x == 0 && P.hctl) P.hctl[AESOFF_CTL_SMEMBASE] = sbase;
        fill_tables(tbase, P.T0, tid, AESOFF_WORKER_WARPS * 32u); /* worker threads only */
        if (P.need_dec) fill_td(tbase, P.T0 + 256, tid, AESOFF_WORKER_WARPS * 32u);
        DBG_MAX(2); /* last CTA has its tables */
        asm volatile("bar.sync 1, %0;" ::"n"(AESOFF_CTA_THREADS) : "memory");
        if (tid == 0) sts_volatile(&c->tables_ready, 1u);
        WorkerParams wp;
        wp.dq_done = P.dq_done;
        wp.hmail = P.hmail;
        wp.dev_done_seq = P.dev_done_seq;
        wp.counters = P.counters;
        worker_loop(wp, c, tbase | (lane * 4u), lane);
        DBG_MIN(6); /* first worker warp leaves */
        DBG_MAX(7); /* last worker warp leaves  */
    }
}

/* ------------------------------------------------------------------------------------------ */
/* host-side launch helper (called by aesoff_runtime.cpp)                                      */
/* ------------------------------------------------------------------------------------------ */
extern "C" int aesoff_launch_engine(const aesoff_params_t *params, int n_ctas, void *stream)
{
    /* per device: the attribute belongs to the function as loaded on the current device */
    cudaError_t e = cudaFuncSetAttribute(aesoff_engine_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)AESOFF_SMEM_BYTES);
    if (e != cudaSuccess) return (int)e;
    const uint32_t smem = params->need_dec ? AESOFF_SMEM_BYTES : AESOFF_SMEM_BYTES_NODEC;
    aesoff_engine_kernel<<<n_ctas, AESOFF_CTA_THREADS, smem, (cudaStream_t)stream>>>(*params);
    return (int)cudaGetLastError();
}

/* ------------------------------------------------------------------------------------------ */
/* aes_ctr_launch_static: the launch backend for callers that must not allocate                */
/* ------------------------------------------------------------------------------------------ */
/* Who this is for.  aes_ctr_launch_batch keeps its queue (counters, descriptors, keys, tickets) in
 * device memory that it obtains with cudaMalloc on first use, frees and re-obtains when a batch
 * outgrows it, and fills through a cudaHostAlloc'ed staging buffer.  Three kinds of user of this
 * library cannot live with that:
 *   - a server that gave the GPU's memory to an allocator of its own when it started (a tensor
 *     framework's caching pool, a database's buffer pool): nothing is left, cudaMalloc answers
 *     "out of memory" although the process holds plenty;
 *   - a process in which some kernel never ends -- this library's own persistent engine on that
 *     GPU is one (include/aesoff.h, aes_engine_start), other people's are others: cudaFree waits
 *     for every kernel on the device, that one included, so the re-allocation above never returns;
 *   - a request handler on a latency budget: cudaMalloc and cudaFree take driver-wide locks and
 *     cost from tens of microseconds to milliseconds, more than the 4 KiB offload they would serve.
 * For them the whole queue of ONE request lives in the array below.  It is part of the library's
 * image: every GPU on which the process loads this library carries its AESOFF_STATIC_BYTES (19.25 KiB)
 * from then until the process ends, whether or not this entry point is ever called.
 *
 * Inside host code `g_static_scratch` is not an address a kernel can use -- it names the host-side
 * shadow of the symbol.  The address on a given GPU comes from cudaGetSymbolAddress, asked once per
 * device with that device current (static_scratch_of); device code, like the set-up kernel, may name
 * the array directly.
 *
 * Layout (offsets in bytes; every part starts on a multiple of 128):
 *      0  counters          AESOFF_CNT_WORDS x 8    rewritten by every call's set-up kernel
 *    512  dq_done           one countdown word       cleared by every call
 *    640  dev_done_seq      one word
 *    768  dq                ONE descriptor (the request), tagged pieces
 *   1024  ktab              ONE expanded key
 *   1280  T0 | Td0          2 KiB, written once per device by static_scratch_of and never again
 *   3328  tmap              AESOFF_STATIC_TICKETS tickets of 16 bytes
 */
#define AESOFF_STATIC_TICKETS 1024u
#define AESOFF_STATIC_OFF_DONE 512u
#define AESOFF_STATIC_OFF_SEQ 640u
#define AESOFF_STATIC_OFF_DQ 768u
#define AESOFF_STATIC_OFF_KEY 1024u
#define AESOFF_STATIC_OFF_T0 1280u
#define AESOFF_STATIC_OFF_TMAP 3328u
#define AESOFF_STATIC_BYTES (AESOFF_STATIC_OFF_TMAP + AESOFF_STATIC_TICKETS * 16u)

static __device__ __align__(256) uint8_t g_static_scratch[AESOFF_STATIC_BYTES];

extern "C" int aesoff_fail(int code);          /* aesoff_runtime.cpp: files the code for aes_last_error() */
extern "C" void aesoff_note_launches(int n);   /* aesoff_runtime.cpp: aes_engine_info_t::kernel_launches   */

namespace {

/* everything the set-up kernel needs, passed by value as its kernel argument (376 bytes) */
struct StaticJob {
    aesoff_dev_desc_t desc; /* the request as the service warps read it */
    uint32_t rk[60];        /* its expanded key                          */
    uint32_t total;         /* tickets = chunks of the request           */
    uint32_t crows;         /* rows per chunk                            */
    uint64_t rows;
    uint64_t wave;          /* rows the grid's worker warps take at once */
};

/* Writes the call's queue into the static array.  The array still holds the previous call's queue, so every
 * word the engine kernel reads before writing is stored here again: all counters (the ticket counter must
 * start at 0), the chunk countdown, the completion word, the descriptor, the key and tickets 0 .. total-1.
 * Tickets past `total` are stale but never reserved (drain_total).                                        */
__global__ void __launch_bounds__(256) aesoff_static_setup_kernel(const StaticJob J)
{
    uint8_t *base = g_static_scratch; /* device code names the array itself */
    const uint32_t tid = threadIdx.x;
    unsigned long long *cnt = reinterpret_cast<unsigned long long *>(base);
    if (tid < AESOFF_CNT_WORDS) cnt[tid] = (tid == AESOFF_CNT_PUBLISHED) ? (unsigned long long)J.total : 0ull;
    if (tid == 64) *reinterpret_cast<uint32_t *>(base + AESOFF_STATIC_OFF_DONE) = 0u;
    if (tid == 65) *reinterpret_cast<unsigned long long *>(base + AESOFF_STATIC_OFF_SEQ) = 0ull;
    if (tid >= 96 && tid < 128) { /* descriptor word p at w[(p / 3) * 4 + p % 3], tag = sequence number 1 */
        const uint32_t i = tid - 96u, q = i >> 2, r = i & 3u;
        const uint32_t *w = reinterpret_cast<const uint32_t *>(&J.desc);
        reinterpret_cast<uint32_t *>(base + AESOFF_STATIC_OFF_DQ)[i] = (r == 3u) ? 1u : w[3u * q + r];
    }
    if (tid >= 128 && tid < 192) {
        const uint32_t i = tid - 128u;
        reinterpret_cast<uint32_t *>(base + AESOFF_STATIC_OFF_KEY)[i] = i < 60u ? J.rk[i] : 0u;
    }
    /* the same end-of-launch rule as aes_ctr_launch_batch: the chunks that hold the last wave of rows are cut
     * into 1/8 rows, the four waves before them into half rows                                              */
    for (uint32_t c = tid; c < J.total; c += blockDim.x) {
        const unsigned long long left = J.rows - (unsigned long long)c * J.crows;
        const uint32_t mode = left <= J.wave ? AESOFF_FLAG_FINE : left <= 5ull * J.wave ? AESOFF_FLAG_HALF : 0u;
        reinterpret_cast<uint4 *>(base + AESOFF_STATIC_OFF_TMAP)[c] =
            make_uint4(1u, c | (mode << AESOFF_TICKET_MODE_SHIFT), 0u, c + 1u);
    }
}

std::mutex g_static_mu;
uint8_t *g_static_ptr[AESOFF_MAX_DEVICES]; /* device address of g_static_scratch on each GPU, once known */
int g_static_sms[AESOFF_MAX_DEVICES];

/* Set-up, once per device, with that device current: asks the runtime where the array lives on THIS GPU and
 * puts the two tables there.  The copy is a synchronous cudaMemcpy: this is why the first call on a device
 * belongs before any stream capture.  Returns NULL on error.                                              */
uint8_t *static_scratch_of(int device)
{
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (g_static_ptr[device]) return g_static_ptr[device];
    int sms = 0, major = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess ||
        cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device) != cudaSuccess || major != 10 || sms <= 0)
        return nullptr;
    uint8_t *ptr = nullptr;
    if (cudaGetSymbolAddress((void **)&ptr, g_static_scratch) != cudaSuccess || !ptr) {
        cudaGetLastError();
        return nullptr;
    }
    if (cudaMemcpy(ptr + AESOFF_STATIC_OFF_T0, aesoff_T0_table(), 512 * 4, cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        return nullptr;
    }
    g_static_sms[device] = sms;
    g_static_ptr[device] = ptr;
    return ptr;
}

} /* namespace */

extern "C" __attribute__((visibility("default"))) int aes_ctr_launch_static(aes_ctx_t *ctx, const uint8_t nonce[16],
                                                                            const void *src, void *dst, size_t len,
                                                                            int device, void *cuda_stream)
{
    if (!ctx || !nonce) return aesoff_fail(AES_E_INVAL);
    if (len > (size_t)AES_STATIC_MAX_BYTES) return aesoff_fail(AES_E_TOOBIG);
    if (len == 0) return AES_OK;
    if (!src || !dst) return aesoff_fail(AES_E_INVAL);
    const uintptr_t s = (uintptr_t)src, d = (uintptr_t)dst;
    if ((s | d) & 15u) return aesoff_fail(AES_E_ALIGN);
    if (s != d && s < d + len && d < s + len) return aesoff_fail(AES_E_OVERLAP);
    if (device < 0 || device >= AESOFF_MAX_DEVICES) return aesoff_fail(AES_E_INVAL);
    aes_engine_info_t info;
    if (aes_engine_info_device(device, &info) == AES_OK && info.running) return aesoff_fail(AES_E_BUSY);

    StaticJob J;
    memset(&J, 0, sizeof(J));
    uint8_t rkb[240];
    const int nr = aes_ctx_round_keys(ctx, rkb); /* host expansion, done once per context */
    if (nr < 0) return nr;
    memcpy(J.rk, rkb, (size_t)16 * (nr + 1));    /* little-endian host: FIPS byte string == little-endian-loaded words */

    /* geometry: rows of 256 counter values aligned on counter byte 15 == 0; chunks of 4 rows, doubled until
     * the request fits the ticket array (64 MiB: 16,385 rows -> 513 chunks of 32)                          */
    const uint64_t nblocks = ((uint64_t)len + 15u) >> 4;
    const uint64_t rows = (nblocks + nonce[15] + AESOFF_ROW_BLOCKS - 1) >> 8;
    uint32_t crows = 4;
    while ((rows + crows - 1) / crows > AESOFF_STATIC_TICKETS) crows *= 2;
    const uint32_t total = (uint32_t)((rows + crows - 1) / crows);

    int ndev = 0, prev = -1;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device >= ndev || cudaGetDevice(&prev) != cudaSuccess) {
        cudaGetLastError();
        return aesoff_fail(AES_E_CUDA);
    }
    if (prev != device && cudaSetDevice(device) != cudaSuccess) {
        cudaGetLastError();
        return aesoff_fail(AES_E_CUDA);
    }
    int rc = AES_OK;
    uint8_t *ptr = static_scratch_of(device);
    if (!ptr) {
        rc = AES_E_CUDA;
    } else {
        memcpy(J.desc.icb, nonce, 16);
        J.desc.src = (uint64_t)s;
        J.desc.dst = (uint64_t)d;
        J.desc.len = (uint64_t)len;
        J.desc.nr = (uint32_t)nr;
        J.desc.flags = AESOFF_MODE_CTR;
        J.desc.nchunks = total;
        J.desc.chunk_rows = crows;
        J.desc.seq = 1;
        J.desc.rows = rows;
        J.desc.first_ticket = 0;
        J.desc.keyloc = 0;
        J.total = total;
        J.crows = crows;
        J.rows = rows;
        J.wave = (uint64_t)g_static_sms[device] * AESOFF_WORKER_WARPS;

        aesoff_params_t p;
        memset(&p, 0, sizeof(p));
        p.counters = reinterpret_cast<uint64_t *>(ptr);
        p.dq_done = reinterpret_cast<uint32_t *>(ptr + AESOFF_STATIC_OFF_DONE);
        p.dev_done_seq = reinterpret_cast<uint64_t *>(ptr + AESOFF_STATIC_OFF_SEQ);
        p.dq = reinterpret_cast<aesoff_dq_entry_t *>(ptr + AESOFF_STATIC_OFF_DQ);
        p.ktab = reinterpret_cast<aesoff_key_t *>(ptr + AESOFF_STATIC_OFF_KEY);
        p.T0 = reinterpret_cast<const uint32_t *>(ptr + AESOFF_STATIC_OFF_T0);
        p.tmap = reinterpret_cast<aesoff_ticket_t *>(ptr + AESOFF_STATIC_OFF_TMAP);
        p.drain_total = total;
        p.R = 1;                       /* one request: every sequence number maps to entry 0 */
        p.TM = AESOFF_STATIC_TICKETS;
        p.chunk_rows = crows;
        p.mode = AESOFF_MODE_DRAIN;
        p.first_seq = 1;
        uint64_t ctas = (rows + AESOFF_ROWS_PER_CTA - 1) / AESOFF_ROWS_PER_CTA;
        if (ctas > (uint64_t)g_static_sms[device]) ctas = (uint64_t)g_static_sms[device];
        cudaStream_t stream = (cudaStream_t)cuda_stream;
        aesoff_static_setup_kernel<<<1, 256, 0, stream>>>(J);
        if (cudaGetLastError() != cudaSuccess || aesoff_launch_engine(&p, (int)ctas, stream) != 0) {
            cudaGetLastError();
            rc = AES_E_CUDA;
        } else {
            aesoff_note_launches(2);
        }
    }
    explicit_bzero(&J, sizeof(J)); /* key hygiene: the expanded key was on this stack frame */
    explicit_bzero(rkb, sizeof(rkb));
    if (prev != device) cudaSetDevice(prev);
    return rc == AES_OK ? AES_OK : aesoff_fail(rc);
}

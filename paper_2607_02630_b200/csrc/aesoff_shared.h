/*
 * aesoff_shared.h -- structures shared by the host runtime and the sm_100a kernels
 * (internal; the public boundary is include/aesoff.h).
 *
 * Data layout in memory:
 *   host ring    pinned, host-mapped, R slots of 384 B.  The host writes the 288-byte
 *                body, then release-stores `seq` (own 64-byte line).     step a2
 *   dq           device memory, R descriptors of 320 B: the body copied by the
 *                dispatcher plus the chunk geometry it derived.           step a3
 *   tmap         device memory ring of 2^k 8-byte tickets (seq << 24 | chunk).
 *   mailbox      pinned, host-mapped, R x 8 B: slot -> last completed seq.  step a7
 */
#ifndef AESOFF_SHARED_H
#define AESOFF_SHARED_H

#include <stdint.h>

#define AESOFF_ROW_BLOCKS      256u   /* counter values per row: one value of the low counter byte each */
#define AESOFF_ROW_BYTES       4096u
#define AESOFF_WORKER_WARPS    16u    /* warps that run the cipher; 4 per SM sub-partition               */
#define AESOFF_SLOTS           16u    /* chunk tickets a CTA holds in shared memory (open + prefetched)   */
#define AESOFF_CTA_THREADS     ((AESOFF_WORKER_WARPS + 2u) * 32u) /* + service warp + dispatcher warp      */
#define AESOFF_ROWS_PER_CTA    16u    /* drain mode: one CTA per this many rows of work, up to the SM count */
#define AESOFF_FLAG_FINE       1u     /* descriptor flag: units of 1/8 row (32 blocks) instead of a row   */
#define AESOFF_FINE_ALWAYS_ROWS 16u   /* requests up to 64 KiB are always cut fine (submission-bound)     */
#define AESOFF_BODY_BYTES      288u
#define AESOFF_DESC_BYTES      320u
#define AESOFF_TICKET_CHUNK_BITS 24u
#define AESOFF_SMEM_BYTES      (192u * 1024u)

#define AESOFF_MODE_PERSISTENT 0u
#define AESOFF_MODE_DRAIN      1u

/* host-mapped control words (uint32 each) */
#define AESOFF_CTL_STOP        0      /* host -> device: 1 = exit after the ring is drained */
#define AESOFF_CTL_ALIVE       1      /* device -> host: 1 once the kernel polls, 2 after it exits */
#define AESOFF_CTL_SMEMBASE    2      /* device -> host: shared-window offset of dynamic smem (debug) */
#define AESOFF_CTL_WORDS       16

/* device counters (index in uint64 units) */
#define AESOFF_CNT_TICKET      0      /* next ticket to hand out (atomicAdd by the service warps)      */
#define AESOFF_CNT_PUBLISHED   1      /* tickets the dispatcher has published; same 16 B as TICKET      */
#define AESOFF_CNT_IDLE        8      /* CTAs of the persistent engine that have no open slot           */
#define AESOFF_CNT_STOP        16
#define AESOFF_CNT_WORDS       32

typedef struct __attribute__((aligned(128))) aesoff_host_slot {
    uint32_t rk[60];       /*   0: round keys, word c of round r at rk[4r+c], little-endian load of the
                                   FIPS-197 byte string (byte 0 of the word = row 0 of column c)      */
    uint32_t icb[4];       /* 240: the 16 counter-block bytes, same loading                            */
    uint64_t src;          /* 256 */
    uint64_t dst;          /* 264 */
    uint64_t len;          /* 272 */
    uint32_t nr;           /* 280: 10 or 14                                                            */
    uint32_t flags;        /* 284 */
    uint64_t pad0[4];      /* 288 */
    volatile uint64_t seq; /* 320: valid flag = the request's sequence number, written last            */
    uint64_t pad1[7];
} aesoff_host_slot_t;      /* 384 bytes */

typedef struct __attribute__((aligned(16))) aesoff_dev_desc {
    uint32_t rk[60];
    uint32_t icb[4];
    uint64_t src;
    uint64_t dst;
    uint64_t len;
    uint32_t nr;
    uint32_t flags;
    /* written by the dispatcher (or by the host for the launch backend) */
    uint32_t nchunks;      /* 288 */
    uint32_t chunk_rows;   /* 292: rows per chunk for this request                                     */
    uint64_t seq;          /* 296 */
    uint64_t rows;         /* 304: number of 256-counter rows the request touches                      */
    uint64_t pad;          /* 312 */
} aesoff_dev_desc_t;       /* 320 bytes */

typedef struct aesoff_params {
    aesoff_host_slot_t *hring;      /* host-mapped (persistent mode)                     */
    volatile uint64_t  *hmail;      /* host-mapped mailbox, may be NULL in drain mode    */
    volatile uint32_t  *hctl;       /* host-mapped control words, NULL in drain mode     */
    aesoff_dev_desc_t  *dq;
    uint64_t           *tmap;
    uint64_t           *counters;
    uint32_t           *dq_done;
    uint64_t           *dev_done_seq;
    const uint32_t     *T0;         /* 256 words: T0[x] = {02}S | S<<8 | S<<16 | {03}S<<24 */
    uint64_t            drain_total;
    uint32_t            R;          /* ring slots, power of two                          */
    uint32_t            TM;         /* ticket ring entries, power of two                 */
    uint32_t            chunk_rows;
    uint32_t            mode;
    uint32_t            idle_exit_ms;
    uint32_t            fine_rows;  /* requests of at most this many rows may be cut into 1/8-row units; 0 = never */
    uint64_t            first_seq;  /* sequence number of the first request of this launch */
} aesoff_params_t;

#endif

/*
 * aesoff_shared.h -- structures shared by the host runtime and the sm_100a kernels
 * (internal; the public boundary is include/aesoff.h).
 *
 * Data layout in memory:
 *   host ring    pinned, host-mapped, R slots of 128 B = 8 self-validating 16-byte pieces
 *                (3 payload words + the low 32 bits of the request's sequence number).  The
 *                host writes each piece with ONE 16-byte store, the dispatcher reads each with
 *                ONE 16-byte load, so a piece is either the old one or the new one and the whole
 *                descriptor arrives in a single PCIe round trip (no flag-then-body).   step a2
 *   dq           device memory, R descriptors of 128 B (96 B of fields as 8 tagged pieces): the
 *                request plus the chunk geometry the dispatcher derived.                step a3
 *   ktab         device memory, (AESOFF_KEY_IDS + R) expanded keys of 256 B: entries below
 *                AESOFF_KEY_IDS belong to contexts that have been installed, the rest to ring
 *                slots (keys of one-shot contexts, expanded on the device).            step a1
 *   tmap         device memory ring of 2^k 16-byte tickets {seq low half, chunk, key index, tag}.
 *   mailbox      pinned, host-mapped, R x 8 B: slot -> last completed seq.             step a7
 */
#ifndef AESOFF_SHARED_H
#define AESOFF_SHARED_H

#include <stdint.h>

#define AESOFF_ROW_BLOCKS      256u   /* counter values per row: one value of the low counter byte each */
#define AESOFF_ROW_BYTES       4096u
#ifndef AESOFF_WORKER_WARPS
#define AESOFF_WORKER_WARPS    16u    /* warps that run the cipher; 4 per SM sub-partition               */
#endif
#define AESOFF_ROWS_PER_UNIT   2u     /* whole-row units (saturation) are this many consecutive rows      */
#ifndef AESOFF_NB
#define AESOFF_NB              4      /* blocks a lane keeps in flight through the rounds (row units)     */
#endif
#define AESOFF_SLOTS           16u    /* chunk tickets a CTA holds in shared memory (open + prefetched)   */
#define AESOFF_CTA_THREADS     ((AESOFF_WORKER_WARPS + 2u) * 32u) /* + service warp + dispatcher warp      */
#define AESOFF_ROWS_PER_CTA    16u    /* drain mode: one CTA per this many rows of work, up to the SM count */
#define AESOFF_FLAG_FINE       1u     /* descriptor flag: units of 1/8 row (32 blocks) instead of a row   */
#define AESOFF_FLAG_HALF       2u     /* descriptor flag: units of half a row (128 blocks)                */
#define AESOFF_FINE_ALWAYS_ROWS 16u   /* requests up to 64 KiB are always cut fine (submission-bound)     */
#define AESOFF_DESC_BYTES      96u
#define AESOFF_KEY_BYTES       256u   /* one ktab entry: 60 round-key words + padding                     */
#define AESOFF_KEY_IDS         4096u  /* ktab entries that installed contexts can own                      */
#define AESOFF_KEY_NONE        0xffffu
#define AESOFF_SMEM_BYTES      (223u * 1024u) /* with the decryption table: control block, 4 encryption tables (128 KiB) on a
                                                 64 KiB boundary of the shared window, Td0 (32 KiB); leaves 4 KiB of the SM */
#define AESOFF_SMEM_BYTES_NODEC (200u * 1024u) /* without Td0: 27 KiB of the SM's shared memory stay free for other kernels */

/* what a request computes (descriptor word `flags`; SP 800-38A sec. 6.5, 6.1, 6.2) */
#define AESOFF_MODE_CTR        0
#define AESOFF_MODE_ECB_ENC    1
#define AESOFF_MODE_ECB_DEC    2
#define AESOFF_MODE_CBC_DEC    3

#define AESOFF_MODE_PERSISTENT 0u
#define AESOFF_MODE_DRAIN      1u

/* host-mapped control words (uint32 each) */
#define AESOFF_CTL_STOP        0      /* host -> device: 1 = exit after the ring is drained */
#define AESOFF_CTL_ALIVE       1      /* device -> host: 1 once the kernel polls, 2 after it exits */
#define AESOFF_CTL_SMEMBASE    2      /* device -> host: shared-window offset of dynamic smem (debug) */
#define AESOFF_CTL_STATS       16     /* device -> host, 8 words per dispatcher warp d at 16 + 8 d (statistics): */
#define AESOFF_CTL_CUT_EIGHTHS 0      /*   requests whose first chunk was cut into 1/8-row units so far          */
#define AESOFF_CTL_CUT_HALVES  1      /*   ... into half rows                                                    */
#define AESOFF_CTL_CUT_ROWS    2      /*   ... into whole rows                                                   */
#define AESOFF_MAX_DISPATCHERS 8u     /* dispatcher warps (warp 17 of CTAs 0 .. n-1); default AESOFF_DEF_DISPATCHERS */
#define AESOFF_DEF_DISPATCHERS 2u
#define AESOFF_BATCH           32u    /* consecutive sequence numbers one dispatcher takes: batch b belongs to dispatcher b % n */
#define AESOFF_CTL_DBG_TAKES   3      /*   (AESOFF_DISP_STATS builds) polls that took requests, ...              */
#define AESOFF_CTL_DBG_REQS    4      /*   ... requests taken, ...                                               */
#define AESOFF_CTL_DBG_WAIT    5      /*   ... time spent waiting for the token, in units of 64 ns, ...          */
#define AESOFF_CTL_DBG_WORK    6      /*   ... time from the token to the last ticket store, in units of 64 ns   */
#define AESOFF_CTL_DBG_EMPTY   7      /*   ... polls that found nothing                                          */
#define AESOFF_CTL_STAT_WORDS  8
#define AESOFF_CTL_WORDS       128

/* device counters (index in uint64 units) */
#define AESOFF_CNT_TICKET      0      /* next ticket to hand out (atomicAdd by the service warps)      */
#define AESOFF_CNT_PUBLISHED   1      /* tickets the dispatcher has published; same 16 B as TICKET      */
#define AESOFF_CNT_IDLE        8      /* CTAs of the persistent engine that have no open slot           */
#define AESOFF_CNT_QUIT        9      /* low half: dispatcher 0 -> the others: leave (idle timer); high half: the dispatcher
                                         that holds the token found a long queue (the others prefetch their batches);
                                         same 16 B as IDLE */
#define AESOFF_CNT_STOP        16
#define AESOFF_CNT_DEBUG       20     /* 8 words of time stamps in AESOFF_DEBUG builds                   */
#define AESOFF_CNT_CHAIN       32     /* {tickets published, next sequence number to dispatch}: the token the
                                         dispatcher warps pass along, one 16-byte word on a line of its own */
#define AESOFF_CNT_WORDS       64

/* ---- host ring slot: 8 pieces of {payload[3], tag}; tag = (uint32_t)seq -------------------- */
/* payload word p (0..23) of a slot is w[(p / 3) * 4 + p % 3]                                    */
#define AESOFF_PW_ICB          0      /* 4 words: the 16 counter-block bytes, little-endian loads   */
#define AESOFF_PW_SRC          4      /* 2 words */
#define AESOFF_PW_DST          6      /* 2 words */
#define AESOFF_PW_LEN          8      /* 2 words */
#define AESOFF_PW_KEY          10     /* key word, see AESOFF_KW_*                                  */
#define AESOFF_PW_SPARE        11     /* AESOFF_MODE_CTR / _ECB_ENC / _ECB_DEC / _CBC_DEC (the ICB words then hold the IV) */
#define AESOFF_PW_RAWKEY       12     /* 8 words (second 64-byte line): the cipher key itself       */
#define AESOFF_PW_WORDS        24
#define AESOFF_PW_INDEX(p)     (((p) / 3) * 4 + (p) % 3)
/* key word: bits 0..15 ktab index of the context (AESOFF_KEY_NONE = none), bit 16 raw key present
 * in the second line (the dispatcher expands it, FIPS-197 sec. 5.2), bit 17 store the expanded key
 * at the ktab index for later requests, bits 24..31 Nr (10 or 14)                                */
#define AESOFF_KW_RAW          (1u << 16)
#define AESOFF_KW_INSTALL      (1u << 17)

typedef struct __attribute__((aligned(128))) aesoff_host_slot {
    uint32_t w[32];
} aesoff_host_slot_t;      /* 128 bytes */

typedef struct __attribute__((aligned(16))) aesoff_dev_desc {
    uint32_t icb[4];       /*  0: the 16 counter-block bytes, little-endian loads                    */
    uint64_t src;          /* 16 */
    uint64_t dst;          /* 24 */
    uint64_t len;          /* 32 */
    uint32_t nr;           /* 40: 10 or 14                                                             */
    uint32_t flags;        /* 44: AESOFF_FLAG_*                                                        */
    uint32_t nchunks;      /* 48 */
    uint32_t chunk_rows;   /* 52: rows per chunk for this request                                      */
    uint64_t seq;          /* 56 */
    uint64_t rows;         /* 64: number of 256-counter rows the request touches                       */
    uint64_t first_ticket; /* 72 */
    uint32_t keyloc;       /* 80: ktab index of the expanded key                                       */
    uint32_t pad[3];
} aesoff_dev_desc_t;       /* 96 bytes */

/* dq entry in device memory: the 24 words of aesoff_dev_desc_t as 8 pieces of {3 words, tag}, tag = low 32
 * bits of the request's sequence number -- self-validating like a host ring slot, so that the dispatcher
 * needs no fence between writing a descriptor and writing the tickets that point at it: a service warp that
 * reads a piece too early sees a wrong tag and reads again.                                              */
typedef struct __attribute__((aligned(128))) aesoff_dq_entry {
    uint32_t w[32];        /* word p (0..23) of the descriptor at w[(p / 3) * 4 + p % 3], tags at w[4q + 3] */
} aesoff_dq_entry_t;       /* 128 bytes */

typedef struct __attribute__((aligned(16))) aesoff_key {
    uint32_t rk[60];       /* round keys, word c of round r at rk[4r+c], little-endian load of the
                              FIPS-197 byte string (byte 0 of the word = row 0 of column c)            */
    uint32_t pad[4];
} aesoff_key_t;            /* 256 bytes */

#define AESOFF_TICKET_CHUNK_MASK 0x0fffffffu
#define AESOFF_TICKET_MODE_SHIFT 28u
typedef struct __attribute__((aligned(16))) aesoff_ticket {
    uint32_t seq32;        /* low 32 bits of the request's sequence number: (seq32 - 1) & (R - 1) is its
                              index in dq / mailbox, and seq32 the tag its dq pieces must carry         */
    uint32_t chunk;        /* bits 0..27 chunk index; bits 28..29 unit size of this chunk:
                              0 rows, AESOFF_FLAG_FINE 1/8 rows, AESOFF_FLAG_HALF half rows            */
    uint32_t keyloc;
    uint32_t tag;          /* (uint32_t)ticket number + 1; the ring is zeroed at engine start          */
} aesoff_ticket_t;         /* 16 bytes, written and read as one 128-bit access                         */

/* unit-size policy of the persistent dispatcher; W = worker warps of the grid */
#define AESOFF_TUNE_FINE_TOTAL   0    /* idle GPU, whole known queue at most this many rows: 1/8-row units (W / 4) */
#define AESOFF_TUNE_FINE_FRONT   1    /* idle GPU: the first this many rows of the queue in 1/8 rows     (0: off) */
#define AESOFF_TUNE_HALF_TOTAL   2    /* known queue at most this many rows: half rows                   (3 W / 4) */
#define AESOFF_TUNE_TAIL_AHEAD   3    /* a request that found at most this many rows ahead of it ...     (W)     */
#define AESOFF_TUNE_TAIL_LEFT    4    /* ... has its last this many rows cut into half rows              (2 W)   */
#define AESOFF_TUNE_SPREAD_AHEAD 5    /* idle GPU and at most this many rows ahead: one chunk per CTA ... (W / 2) */
#define AESOFF_TUNE_SPREAD_MAX   6    /* ... of at most this many rows                                   (16)    */
#define AESOFF_TUNE_POLL_DEPTH   7    /* polls of the ring the token holder keeps in flight while the queue is short (1..3) */
#define AESOFF_TUNE_PRERESERVE   9    /* a CTA holding less than this many 1/8 rows per worker keeps a reservation on a ticket that does not exist yet */
#define AESOFF_TUNE_POLL_GAP     8    /* nanoseconds between issuing them, so that they stay spread over a round trip       */

typedef struct aesoff_params {
    aesoff_host_slot_t *hring;      /* host-mapped (persistent mode)                     */
    volatile uint64_t  *hmail;      /* host-mapped mailbox, may be NULL in drain mode    */
    volatile uint32_t  *hctl;       /* host-mapped control words, NULL in drain mode     */
    aesoff_dq_entry_t  *dq;
    aesoff_key_t       *ktab;
    aesoff_ticket_t    *tmap;
    uint64_t           *counters;
    uint32_t           *dq_done;
    uint64_t           *dev_done_seq;
    const uint32_t     *T0;         /* 256 words: T0[x] = {02}S | S<<8 | S<<16 | {03}S<<24; then 256 words Td0 */
    uint32_t            need_dec;   /* fill the Td0 table (always in persistent mode; drain: a decrypt request in the batch) */
    uint64_t            drain_total;
    uint32_t            R;          /* ring slots, power of two                          */
    uint32_t            TM;         /* ticket ring entries, power of two                 */
    uint32_t            chunk_rows;
    uint32_t            chunk_log2; /* chunk_rows == 1 << chunk_log2 */
    uint32_t            mode;
    uint32_t            idle_exit_ms;
    uint32_t            fine_rows;  /* requests of at most this many rows may be cut into units smaller than a row; 0 = never */
    uint64_t            first_seq;  /* sequence number of the first request of this launch */
    uint32_t            n_disp;     /* dispatcher warps (persistent mode), 1 .. AESOFF_MAX_DISPATCHERS      */
    uint32_t            tune[10];    /* dispatcher policy, AESOFF_TUNE_* (dispatcher_loop)                   */
} aesoff_params_t;

#endif

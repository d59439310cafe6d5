/*
 * aesoff.h -- C ABI of the B200 AES-CTR offload engine.
 *
 * What this library is.  The paper's servers reroute one fine-grained routine to
 * an accelerator: `accel_encrypt(j.buf, j.len)` (Listing 1), which
 * "performs AES ... on its own CUDA stream, polled by cudaEventQuery, with the
 * block size sweeping from 4 KiB (launch-bound) to 8 MiB (bandwidth-bound)"
 * (section 6 "Experimental setup").  The calls below are that
 * routine split along the paper's three-step recipe (section 3:
 * "submit the work to a background executor instead of waiting", "suspend the
 * current request", "resume it ... when the offload completes"):
 *
 *     submit  -> aes_ctr_submit()   returns a completion handle at once
 *     suspend -> the caller's job (suspend BEFORE submitting)
 *     resume  -> the caller's executor spins on aes_poll() / aes_wait()
 *
 * The paper fixes neither mode nor key size; BASELINE.json fixes AES-128 and
 * AES-256 in CTR mode (SP 800-38A sec. 6.5 over FIPS-197), DESIGN.md lists every
 * such reading.  No floating point anywhere: results are exact and unique.
 *
 * Conventions common to all calls
 *   - Plain C types only.  "host" / "device" is stated for every pointer.
 *   - One engine per GPU, up to 8 per process (one process per GPU works as well).  All calls are thread-safe
 *     unless stated; aes_ctr_submit() may be called from many executor threads
 *     ("worker pool", "32-thread executor").
 *   - Errors are negative ints (AES_E_*); a call that returns NULL / 0 leaves
 *     the code in a thread-local slot read by aes_last_error().  Nothing aborts,
 *     nothing throws.  There is NO CPU fallback: without a CUDA device every
 *     compute call fails with AES_E_CUDA.
 *   - Key hygiene and side channels.  aes_ctx_destroy wipes the context; ring slots,
 *     the device key table and the launch backend's staging blob are wiped when they
 *     are freed.  The cipher is table based (T-tables in shared memory, FIPS-197
 *     sec. 5.1 folded): its memory access pattern depends on key and data, as in
 *     every table-based AES.  Each lane reads only its own bank, so there are no
 *     data-dependent bank conflicts inside a warp, but this is NOT a constant-time
 *     implementation and must not share a GPU with an adversary that can time it.
 */
#ifndef AESOFF_H
#define AESOFF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif
#if defined(__GNUC__)
#pragma GCC visibility push(default)   /* the library itself is built with -fvisibility=hidden */
#endif

/* ---- error codes ---------------------------------------------------------- */
#define AES_OK           0
#define AES_E_INVAL     -1   /* NULL pointer, bad option value                      */
#define AES_E_KEYBITS   -2   /* keybits not 128, 192 or 256                        */
#define AES_E_ALIGN     -3   /* src or dst not 16-byte aligned                     */
#define AES_E_OVERLAP   -4   /* src/dst overlap partially (dst == src is allowed)  */
#define AES_E_AGAIN     -5   /* submission ring full: retry after some completions */
#define AES_E_TIMEOUT   -6   /* aes_wait() timed out                               */
#define AES_E_STOPPED   -7   /* engine not running (never started, stopped, dead)  */
#define AES_E_CUDA      -8   /* a CUDA runtime call failed / no device             */
#define AES_E_BUSY      -9   /* call not allowed while the engine is running       */
#define AES_E_NOMEM     -10  /* host or device allocation failed                   */
#define AES_E_TOOBIG    -11  /* aes_ctr_launch_static: len > AES_STATIC_MAX_BYTES   */

/* what a request computes (SP 800-38A sec. 6.5, 6.1, 6.2) */
#define AES_MODE_CTR     0
#define AES_MODE_ECB_ENC 1
#define AES_MODE_ECB_DEC 2
#define AES_MODE_CBC_DEC 3

typedef struct aes_ctx aes_ctx_t;     /* opaque; owns a copy of the expanded round keys */
typedef uint64_t       aes_handle_t;  /* submission sequence number, from 1; 0 = invalid */

/* ---- engine life cycle (step a0 of the path) -------------------------------
 * The engine is: a pinned, host-mapped descriptor ring; ONE persistent sm_100a
 * kernel (dispatcher warps that poll the ring over PCIe, and per SM one
 * service warp plus 16 worker warps around the AES tables in shared memory);
 * and a host-mapped completion
 * mailbox.  A request therefore never pays a kernel launch (the paper's 4 KiB
 * point is "launch-bound").                                       */
#define AES_FINE_ROWS_OFF 0xffffffffu
typedef struct aes_engine_opts {
    uint32_t ring_slots;      /* descriptor ring depth = max requests in flight; power of
                                 two in [64, 4096]; 0 = default 2048                      */
    uint32_t chunk_rows;      /* work-item size in 4 KiB rows (256 counter values each): a power
                                 of two, 1..64; 0 = default 4 (16 KiB per worker-group item) */
    uint32_t n_ctas;          /* persistent CTAs; 0 = one per SM                          */
    uint32_t idle_exit_ms;    /* the kernel exits by itself (engine becomes STOPPED) after
                                 this long with no request; 0 = never                     */
    uint32_t fine_rows;       /* latency modes: a request of at most this many 4 KiB rows may
                                 be cut into units smaller than a row -- 1/8 row (32 blocks per
                                 warp) at the front of an idle GPU's queue, half a row while the
                                 queue is short and at the end of a long lone request -- so that
                                 it spreads over many warps.  0 = default (any size),
                                 AES_FINE_ROWS_OFF = whole rows only                        */
    uint32_t n_dispatchers;   /* warps that poll the ring and cut requests into work items, one
                                 each on the first CTAs; consecutive batches of 32 sequence
                                 numbers go round them.  1..8; 0 = default 2               */
    uint32_t flags;           /* AES_ENGINE_* bits                                        */
    uint32_t reserved[1];     /* must be 0                                                */
} aes_engine_opts_t;
/* Leave the decryption table out: aes_ecb_submit(decrypt) and aes_cbc_decrypt_submit then fail with AES_E_INVAL, and
 * each persistent CTA takes 200 KiB of its SM's shared memory instead of 223 KiB, so that kernels of the process's own
 * that need up to 27 KiB of shared memory per CTA can run beside the engine (with the table: up to 3 KiB).         */
#define AES_ENGINE_NO_DECRYPT 1u

/* Starts the engine on CUDA device `device`.  opts == NULL means all defaults.
 * Returns AES_OK, AES_E_BUSY if already running, AES_E_INVAL, AES_E_CUDA, AES_E_NOMEM.
 * While the engine runs, a device-wide synchronisation (cudaDeviceSynchronize,
 * cudaFree, torch.cuda.synchronize) blocks until aes_engine_stop(): synchronise
 * on streams or events instead.  Copies and other kernels run beside the engine
 * (it leaves 1,472 threads, 10 K registers and a few KiB of shared memory per SM -- see AES_ENGINE_NO_DECRYPT --),
 * with one catch: the FIRST
 * launch of a kernel whose module CUDA has not loaded yet (lazy loading) blocks
 * until the engine stops -- launch every kernel once before aes_engine_start, or
 * run with CUDA_MODULE_LOADING=EAGER.
 * The persistent engine cannot run under a tool that serialises launches (ncu,
 * compute-sanitizer, CUDA_LAUNCH_BLOCKING=1): the launch call then waits for a
 * kernel that waits for submissions.  With idle_exit_ms set the kernel leaves by
 * itself and this call returns AES_E_STOPPED (never AES_OK for an engine that has
 * already exited); with idle_exit_ms == 0 it would not return.  Profile through
 * aes_ctr_launch_batch (the same worker code as an ordinary launch).              */
int aes_engine_start(int device, const aes_engine_opts_t *opts);

/* Refuses new submissions, lets the aes_ctr_submit calls already past that check
 * finish publishing, waits for every accepted request to complete and makes the
 * persistent kernel exit.  Ring and mailbox are kept for the next start.  Handles
 * issued before a clean stop keep answering aes_poll() == 1; if the kernel had died
 * (AES_E_STOPPED is returned) the requests it never completed answer AES_E_STOPPED.
 * Returns AES_OK or AES_E_STOPPED / AES_E_CUDA.                                     */
int aes_engine_stop(void);

typedef struct aes_engine_info {
    int32_t  running;            /* 1 while the persistent kernel is alive           */
    int32_t  device;
    int32_t  sm_count;
    int32_t  n_ctas;
    int32_t  threads_per_cta;
    int32_t  worker_warps_per_cta; /* warps that run the cipher (the rest: service, dispatcher) */
    uint32_t ring_slots;
    uint32_t chunk_rows;
    uint32_t smem_bytes_per_cta;
    uint32_t n_dispatchers;      /* dispatcher warps of the running engine            */
    uint64_t submitted;          /* requests accepted so far                         */
    uint64_t completed;          /* requests whose completion the host has observed
                                    through aes_poll/aes_wait, lower bound            */
    uint64_t kernel_launches;    /* CUDA kernels this library launched so far         */
    uint64_t cut_eighths;        /* requests of the current run the dispatcher cut into
                                    1/8-row units, ...                                */
    uint64_t cut_halves;         /* ... into half rows, ...                           */
    uint64_t cut_rows;           /* ... into whole rows (see fine_rows above)         */
    uint32_t engines_running;    /* engines of this process that accept requests      */
    uint32_t reserved1;
} aes_engine_info_t;
int aes_engine_info(aes_engine_info_t *out);     /* host pointer; AES_OK / AES_E_INVAL.  The running
                                                    engine on the lowest device (else the last one run) */
int aes_engine_info_device(int device, aes_engine_info_t *out);

/* ---- several GPUs: one engine each, and a router ----------------
 * Requests are independent ("each offload belongs to one request"), so the path
 * shards over the GPUs of a node with NO exchange step: aes_engine_start() may be called once per device
 * (up to 8 per process), and aes_ctr_submit() sends each request to the engine of the GPU that owns its
 * device buffer(s) (cudaPointerGetAttributes on src and dst, remembered per 2 MiB page and per thread);
 * requests whose src and dst are both host memory go round the running engines.  A request whose memory
 * belongs to a GPU without a running engine fails with AES_E_STOPPED -- also when only one engine runs on a
 * node with several GPUs.  A request whose src belongs to one GPU and whose dst to another fails with
 * AES_E_INVAL: the engine's kernel would have to dereference a peer pointer, and this library never enables
 * peer access.  Only on a node with ONE GPU is nothing looked up.  A
 * handle carries its engine in its top byte; aes_poll / aes_wait take handles of any engine.  A context
 * may be used on all engines (its key is filed per engine).  NVLink is not used, no collective runs.
 * aes_engine_stop() stops every running engine, aes_engine_stop_device() one.  aes_route_flush() forgets
 * the remembered owners: call it after device memory has been freed and its addresses handed to another GPU. */
int  aes_engine_stop_device(int device);
void aes_route_flush(void);

/* ---- key expansion (step a1; FIPS-197 sec. 5.2) -----------------------------
 * key: host pointer to keybits/8 bytes, copied.  keybits in {128, 192, 256} (BASELINE.json
 * asks for 128 and 256; 192 costs nothing more: Nk = 6, Nr = 12).
 * Returns NULL on error (AES_E_INVAL, AES_E_KEYBITS, AES_E_NOMEM).  Needs no GPU and
 * no running engine; cheap enough to sit on the request path (BASELINE.json
 * configs[3] creates one ctx per request).  Where the expansion itself runs: on the
 * DEVICE for the engine -- the first two submits of a ctx carry the raw key in their
 * descriptor and the dispatcher warp expands it; the second also files the result in
 * a device-side key table, which later submits only name -- and on the host, on
 * demand, for aes_ctx_round_keys and the launch backend.  The key travels with the
 * request, so a ctx may be destroyed as soon as its last submit has returned.      */
aes_ctx_t *aes_ctx_create(const uint8_t *key, int keybits);
void       aes_ctx_destroy(aes_ctx_t *ctx);      /* NULL is a no-op */

/* Copies the 16*(Nr+1) round-key bytes (FIPS-197 byte order: round key r is
 * bytes 16r..16r+15) to `out` (host, >= 240 bytes) and returns Nr (10, 12 or 14), or
 * AES_E_INVAL.  Exists so that tests can pin the key schedule on its own.         */
int aes_ctx_round_keys(const aes_ctx_t *ctx, uint8_t *out);

/* ---- submit (steps a2..a6; SP 800-38A sec. 6.5) -----------------------------
 * Encrypts (= decrypts) len bytes: dst[i] = src[i] xor O[i], where O is the
 * concatenation of Cipher_K(T_1), Cipher_K(T_2), ... with T_1 = nonce and
 * T_{j+1} = (T_j + 1) mod 2^128 read as a big-endian integer; a final partial
 * block uses the leading len mod 16 bytes of its O_n.  No padding.
 *
 *   ctx    host; the key (raw, or the index of its installed expansion) is copied into the descriptor before this returns.
 *   nonce  host; the FULL 16-byte initial counter block T_1 (BASELINE.json
 *          configs[0]: 8-byte nonce || 8-byte big-endian counter from 0); copied.
 *   src    DEVICE pointer on the engine's GPU, or pinned host memory that the GPU
 *          can address (cudaHostAlloc / aes_host_alloc: the kernel then reads it
 *          over PCIe).  16-byte aligned.  Must stay valid and unchanged until
 *          completion.
 *   dst    same kinds of memory, 16-byte aligned, len bytes.  dst == src (in
 *          place) is allowed; any other overlap is AES_E_OVERLAP.
 *   len    any value >= 0 and < 2^36 (64 GiB); len == 0 completes without touching memory.
 *
 * Never blocks.  Returns the handle (>= 1), or 0 with aes_last_error() in
 * {AES_E_INVAL (also: src and dst on two different GPUs), AES_E_ALIGN, AES_E_OVERLAP, AES_E_AGAIN (ring full),
 * AES_E_STOPPED (also: the GPU that owns the memory runs no engine)}.
 * Requests may complete out of order.                                            */
aes_handle_t aes_ctr_submit(aes_ctx_t *ctx, const uint8_t nonce[16],
                            const void *src, void *dst, size_t len);

/* ---- other modes on the same engine ------------------------------------
 * "The GPU path performs AES" with the mode unstated; BASELINE.json fixes CTR for the headline, and
 * the two other modes whose blocks are independent -- so that they spread over warps exactly like CTR -- ride the
 * same ring, units and completion path:
 *   aes_ecb_submit          SP 800-38A sec. 6.1: C_j = Cipher_K(P_j), or with decrypt != 0 P_j = InvCipher_K(C_j)
 *   aes_cbc_decrypt_submit  SP 800-38A sec. 6.2: P_j = InvCipher_K(C_j) xor C_{j-1}, C_0 = iv (host, 16 bytes, copied)
 * (CBC encryption chains every block on the one before it: no data parallelism, not offered.)  Arguments as for
 * aes_ctr_submit, and: len must be a multiple of 16 (AES_E_INVAL; these modes have no partial block, padding is the
 * caller's); for CBC dst must not be src (AES_E_OVERLAP): a block's predecessor is read by another warp, which must
 * find ciphertext there.  Decryption runs the equivalent inverse cipher (FIPS-197 sec. 5.3.5) out of one more
 * table; it is bound by the ALU pipe at about half the CTR rate.                                       */
aes_handle_t aes_ecb_submit(aes_ctx_t *ctx, int decrypt, const void *src, void *dst, size_t len);
aes_handle_t aes_cbc_decrypt_submit(aes_ctx_t *ctx, const uint8_t iv[16], const void *src, void *dst, size_t len);

/* ---- completion (step a7) ----------------------------------------------------
 * aes_poll: 1 = complete, 0 = pending, < 0 = error (AES_E_INVAL for a handle that
 * was never issued, AES_E_STOPPED if the engine died with the request pending).
 * Wait-free: one acquire load of the host-mapped mailbox.  Once it has returned 1,
 * every byte of dst is visible to any copy or kernel issued afterwards on any
 * stream of the device, and to the host if dst is host memory.
 * aes_wait: polls for at most timeout_ns (UINT64_MAX = forever): busy (pause) for the
 * first ~20 us -- the offloads this engine is built for take 10 -- then yielding the
 * core, then sleeping in steps that grow to 50 us, so that a pool of executor threads
 * waiting on long requests does not burn a core each.
 * Returns AES_OK, AES_E_TIMEOUT or the aes_poll error.                             */
int aes_poll(aes_handle_t h);
int aes_wait(aes_handle_t h, uint64_t timeout_ns);

int         aes_last_error(void);          /* thread-local; AES_OK if none          */
const char *aes_strerror(int code);        /* static string                         */

/* ---- launch backend: the paper's own mechanism, for comparison and profiling --
 * "on its own CUDA stream, polled by cudaEventQuery".  Enqueues, on
 * `cuda_stream` (a cudaStream_t passed as void*; NULL = the legacy default
 * stream), one host->device copy of n descriptors followed by ONE ordinary launch
 * of the same worker code the persistent engine runs, which processes the n
 * requests and exits.  Returns after enqueueing; the caller synchronises the
 * stream or an event.  Arrays are host pointers of n entries (nonces: 16*n
 * bytes); src/dst entries as for aes_ctr_submit.  ctxs[i] may repeat.  The
 * persistent engine must NOT be running (its CTAs hold the shared memory):
 * AES_E_BUSY.  chunk_rows as in aes_engine_opts_t (0 = default).  An ordinary
 * launch is what `ncu` can replay, so the committed profiles use this call.       */
int aes_ctr_launch_batch(aes_ctx_t *const *ctxs, const uint8_t *nonces,
                         const void *const *srcs, void *const *dsts,
                         const size_t *lens, size_t n,
                         int device, void *cuda_stream, uint32_t chunk_rows);

/* The same with a mode per request (modes == NULL: all CTR); nonces[16 i ..] is the ICB (CTR), the IV (CBC) or
 * ignored (ECB).  Restrictions of the modes as above.                                                              */
int aes_mode_launch_batch(const int32_t *modes, aes_ctx_t *const *ctxs, const uint8_t *nonces,
                          const void *const *srcs, void *const *dsts,
                          const size_t *lens, size_t n,
                          int device, void *cuda_stream, uint32_t chunk_rows);

/* ---- launch backend without allocation -----------------------------------------------------------
 * aes_ctr_launch_batch obtains its device-side queue with cudaMalloc (and frees / re-obtains it when a batch
 * outgrows it) and a staging buffer with cudaHostAlloc.  Some users of this library cannot do that:
 *   - a server that handed all device memory to a pool of its own at start-up (a tensor framework's caching
 *     allocator, a database's buffer pool): cudaMalloc fails there although the process owns the memory;
 *   - a process with a kernel that never exits on that GPU (this library's persistent engine is one such
 *     kernel; see aes_engine_start): cudaFree waits for it, i.e. for ever;
 *   - a request handler that cannot afford the driver-wide lock and the tens of microseconds to milliseconds
 *     a cudaMalloc / cudaFree costs in front of a 4 KiB offload.
 * aes_ctr_launch_static is the launch backend for ONE CTR request (SP 800-38A sec. 6.5; the offload of
 * PAPER.md:132, on the caller's stream as in PAPER.md:224) that allocates nothing, on the host or on the device:
 * its queue -- counters, one descriptor, one expanded key, the tables, up to 1,024 chunk tickets -- lives in a
 * 19.25 KiB array that is part of the library's image.  Every GPU on which the process loads the library holds
 * that array until the process exits, used or not.  The request and its expanded key travel as the argument of a
 * small set-up kernel; a second launch, the engine kernel in drain mode, does the work.  Both are enqueued on
 * `cuda_stream` (a cudaStream_t of `device`, NULL = the legacy default stream); the call returns after
 * enqueueing and the caller synchronises the stream or an event, as with aes_ctr_launch_batch.
 *
 *   ctx, nonce      host, as for aes_ctr_submit (nonce = the full 16-byte initial counter block).
 *   src, dst        the caller's buffers, as for aes_ctr_submit: memory of `device`, or pinned host memory it can
 *                   address; 16-byte aligned; dst == src allowed.  This call never owns or copies them.
 *   len             0 .. AES_STATIC_MAX_BYTES (64 MiB).  More is refused with AES_E_TOOBIG and nothing is
 *                   enqueued: the ticket array cannot grow.  Split a larger payload into pieces with the counter
 *                   advanced by len / 16 per piece, or use aes_ctr_launch_batch.
 *
 * The first call on each device asks the CUDA runtime for the array's address on that GPU and copies the 2 KiB
 * of tables into it with a synchronous cudaMemcpy; make that first call (len = 16 will do) while the process
 * sets up, before any stream capture begins.  Later calls only launch.  The caller's current device is
 * restored before returning.
 *
 * All calls on a device share the one array, and each call's set-up kernel rewrites the parts that the engine
 * kernel expects to find zeroed or filled (ticket counter, countdown, descriptor, key, tickets) -- so two calls
 * whose kernels can overlap on the GPU (different streams with no dependency between them) corrupt each other's
 * queue.  Keep this entry point's calls on one stream per device, or order them with events.  Calls on the same
 * stream may follow each other without any synchronisation in between.  The persistent engine must not be
 * running on `device` (AES_E_BUSY: its CTAs hold the shared memory).
 * Returns AES_OK, AES_E_INVAL, AES_E_ALIGN, AES_E_OVERLAP, AES_E_TOOBIG, AES_E_BUSY or AES_E_CUDA.             */
#define AES_STATIC_MAX_BYTES (64u << 20)
int aes_ctr_launch_static(aes_ctx_t *ctx, const uint8_t nonce[16], const void *src, void *dst, size_t len,
                          int device, void *cuda_stream);

/* ---- pinned host memory the GPU can address (for host-resident payloads) ----- */
void *aes_host_alloc(size_t bytes);        /* NULL on error (AES_E_CUDA / AES_E_NOMEM) */
void  aes_host_free(void *p);
/* The same for memory the caller already owns -- the paper's request buffer is the server's own (j.buf,
 * PAPER.md:132): page-locks [ptr, ptr + bytes) in place (cudaHostRegister, mapped and portable) so that it may be
 * passed as src / dst of a submit at its own address (16-byte alignment of what is submitted still applies).
 * Registration costs tens of microseconds per MiB: register a server's buffer pool once, not each request, and
 * unregister only after the requests that use the range have completed.  AES_OK, AES_E_INVAL (NULL, zero bytes, already registered),
 * AES_E_NOMEM, AES_E_CUDA.                                                                                      */
int   aes_host_register(void *ptr, size_t bytes);
int   aes_host_unregister(void *ptr);

/* ---- closed-loop executor (the paper's worker pool) ----
 * Drives the running engine from native code so that a microsecond offload is not
 * measured through an interpreter: keeps `window` requests in flight ("submit the
 * next on each completion"), one submitter thread that also polls, and records
 * per-request submit->completion-observed latency.  With keys != NULL a fresh ctx
 * is created (key expansion) and destroyed per request INSIDE the timed loop
 * (BASELINE.json configs[3]); otherwise ctx is shared.  All arrays are host
 * pointers with n entries (nonces: 16*n bytes; keys: 32*n bytes, 16 used when
 * keybits[i] == 128).  lat_ns may be NULL.  `repeat` runs the n requests that many
 * times back to back in one timed region (>= 1).                                   */
typedef struct aes_loop_spec {
    size_t              n;
    uint32_t            window;
    uint32_t            repeat;
    aes_ctx_t          *ctx;        /* shared ctx, used when keys == NULL            */
    const uint8_t      *keys;       /* optional per-request raw keys, 32-byte stride */
    const int32_t      *keybits;    /* with keys: 128, 192 or 256 per request        */
    const uint8_t      *nonces;
    const void *const  *srcs;
    void *const        *dsts;
    const size_t       *lens;
    uint32_t            mode;       /* AES_MODE_CTR (0, the default), _ECB_ENC, _ECB_DEC, _CBC_DEC: what every request of
                                       the run computes; nonces then hold the IVs (CBC) or are ignored (ECB)          */
    uint32_t            reserved;   /* 0 */
} aes_loop_spec_t;

typedef struct aes_loop_result {
    uint64_t elapsed_ns;       /* first submit -> last completion observed           */
    uint64_t bytes;            /* payload bytes completed                             */
    uint64_t requests;         /* requests completed (n * repeat)                     */
    uint64_t ring_full_spins;  /* times submit returned AES_E_AGAIN                   */
    uint64_t max_in_flight;
} aes_loop_result_t;

/* Returns AES_OK or the first error.  lat_ns: host, n*repeat doubles or NULL.      */
int aes_loop_run(const aes_loop_spec_t *spec, aes_loop_result_t *res, double *lat_ns);

/* The same from `nthreads` executor threads (1..64) at once: the n requests are split into
 * contiguous shares, the window is divided among the threads, every thread runs the loop above
 * on its share against the one shared ring.  With repeat > 1, lat_ns holds each thread's share
 * back to back.  elapsed_ns is the wall time of all threads; max_in_flight the sum over threads. */
int aes_loop_run_mt(const aes_loop_spec_t *spec, uint32_t nthreads, aes_loop_result_t *res, double *lat_ns);

/* ---- calibration ---------------------------
 * Runs microkernels with the engine's own table layout and launch shape and reports what the
 * units the cipher leans on deliver on this GPU: table lookups (PRMT + conflict-free LDS.32) per
 * clock per SM, warp-wide ALU instructions (PRMT / LOP3) per clock per SM, the lookup rate of the
 * cipher's main round as it stands, and the GB/s (read + write) of 128-bit L2-only loads and
 * stores over 2 x 1 GiB.  Not on the product path: bench.py and
 * the tests call it.  The engine must not be running (AES_E_BUSY).  Returns AES_OK / AES_E_CUDA.   */
typedef struct aes_calib {
    double  lookups_per_clk_per_sm;      /* nominal 32 (128 B/clk/SM)                         */
    double  alu_instr_per_clk_per_sm;    /* warp-wide; nominal 2 (64 lanes/clk/SM)            */
    double  copy_gbs;
    double  sm_mhz;                      /* SM clock seen by the lookup run                   */
    int32_t sm_count;
    int32_t reserved;
    double  round_lookups_per_clk_per_sm; /* lookups per clock per SM of the cipher's own main
                                             round (4 PRMT + 4 LDS + 2 LOP3 per column): what the
                                             two pipes deliver together                        */
    double  bitslice_sboxes_per_clk_per_sm; /* the alternative to tables: warp-wide evaluations of a bitsliced
                                             S-box (32 lanes x 32 bytes each) per clock per SM  */
    int32_t bitslice_mismatches;         /* of that circuit against S[x] over all 256 inputs: must be 0  */
    int32_t reserved2;
} aes_calib_t;
int aes_calibrate(int device, aes_calib_t *out);

/* ---- open-loop executor (the paper's latency-under-load experiment, Fig. 12) ----
 * Request i arrives arrival_ns[i] nanoseconds after the call starts (host array of spec->n
 * non-decreasing offsets; the caller draws them, e.g. Poisson) and is submitted as soon as that
 * time has passed, whatever is still in flight.  blocking == 0: the loop goes on serving arrivals
 * and polls completions in between (the rerouted server); blocking != 0: it waits for each offload
 * before it looks at the next arrival (the server the paper starts from).  lat_ns[i] = completion
 * observed - arrival time, so queueing in front of a busy loop counts.  spec->ctx is required
 * (keys, window and repeat are ignored).  Returns AES_OK or the first error.                     */
int aes_openloop_run(const aes_loop_spec_t *spec, const uint64_t *arrival_ns, int blocking,
                     aes_loop_result_t *res, double *lat_ns);

#if defined(__GNUC__)
#pragma GCC visibility pop
#endif
#ifdef __cplusplus
}
#endif
#endif /* AESOFF_H */

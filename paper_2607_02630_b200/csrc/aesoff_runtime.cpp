/*
 * aesoff_runtime.cpp -- host runtime behind include/aesoff.h: engine life cycle, the multi-producer
 * submission ring (step a2), the completion mailbox (step a7), the launch backend and the
 * closed-loop executor.  Follows the paper's statement of the problem:
 * submit returns at once, the caller suspends, an executor polls and resumes.
 *
 * Memory-model contract with the kernel (aesoff_kernels.cu):
 *   host: each 16-byte piece of a slot (3 payload words + tag = low half of seq) is written with
 *         ONE 16-byte store                                GPU: reads pieces with 16-byte loads; a
 *         descriptor is taken when all its pieces carry the expected tag (one PCIe round trip)
 *   GPU : dst stores; bar; leader fence.sys; store mailbox  host: acquire-load mailbox[slot] >= seq
 * A slot is reused for seq + R only after mailbox[slot] >= seq has been observed by the submitter.
 */
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <sched.h>
#include <time.h>

#include <algorithm>
#include <atomic>
#include <deque>
#include <mutex>
#include <thread>
#include <vector>

#if defined(__x86_64__)
#include <immintrin.h>
#define CPU_RELAX() _mm_pause()
/* one 16-byte store: a piece of a ring slot is never seen half written */
static inline void store_piece(uint32_t *dst, uint32_t a, uint32_t b, uint32_t c, uint32_t tag)
{
    _mm_store_si128(reinterpret_cast<__m128i *>(dst), _mm_set_epi32((int)tag, (int)c, (int)b, (int)a));
}
#else
#define CPU_RELAX() ((void)0)
static inline void store_piece(uint32_t *dst, uint32_t a, uint32_t b, uint32_t c, uint32_t tag)
{
    unsigned __int128 v = ((unsigned __int128)tag << 96) | ((unsigned __int128)c << 64) | ((unsigned __int128)b << 32) | a;
    __atomic_store_n(reinterpret_cast<unsigned __int128 *>(dst), v, __ATOMIC_RELEASE);
}
#endif

#include "../../include/aesoff.h"
#include "aesoff_internal.h"

namespace {

thread_local int t_last_error = AES_OK;
/* executor threads spread over the shards of per-thread counters */
inline int thread_shard()
{
    static std::atomic<int> next{0};
    thread_local int mine = next.fetch_add(1, std::memory_order_relaxed);
    return mine & 15;
}
inline int fail(int code)
{
    t_last_error = code;
    return code;
}

inline uint64_t now_ns()
{
    struct timespec ts;
    clock_gettime(CLOCK_MONOTONIC_RAW, &ts);
    return (uint64_t)ts.tv_sec * 1000000000ull + (uint64_t)ts.tv_nsec;
}

constexpr int SUBMIT_SHARDS = 16;
struct alignas(64) SubmitShard {
    std::atomic<int> n{0};
};

struct Engine {
    /* Cache-line hygiene for executor pools (32 threads): next_seq is claimed by every submit, so
     * it sits on a line of its own; what every submit and poll only READS (geometry, pointers, running,
     * done_upto) never shares a line with it; the in-flight count is sharded by thread.                   */
    alignas(64) std::atomic<int> running{0};
    int device = -1;
    int sm_count = 0;
    int n_ctas = 0;
    uint32_t n_disp = 1;
    bool has_dec = true;                  /* the decryption table is in shared memory */
    uint32_t R = 0, Rm = 0, chunk_rows = 0, TM = 0;
    cudaStream_t stream = nullptr;
    aesoff_host_slot_t *hring = nullptr; /* pinned, mapped */
    uint64_t *hmail = nullptr;           /* pinned, mapped */
    uint32_t *hctl = nullptr;            /* pinned, mapped */
    aesoff_dq_entry_t *dq = nullptr;
    aesoff_key_t *ktab = nullptr;
    aesoff_ticket_t *tmap = nullptr;
    uint64_t *counters = nullptr, *dev_done_seq = nullptr;
    uint32_t *dq_done = nullptr, *dT0 = nullptr;
    uint64_t first_seq = 1;               /* first sequence number of the current run          */
    alignas(64) std::atomic<uint64_t> next_seq{1}; /* next sequence number to hand out (never reset) */
    alignas(64) SubmitShard submitters[SUBMIT_SHARDS];
    /* ktab indices for installed contexts.  An index freed while next_seq == s is handed out again
     * only once next_seq >= s + R: by then every request that could name it has completed (a ring
     * slot is reused only after its previous request completed).                                  */
    alignas(64) std::mutex id_mu;
    std::deque<std::pair<uint32_t, uint64_t>> id_free; /* (index, next_seq when freed), FIFO   */
    std::atomic<uint64_t> k_epoch{1};     /* bumped whenever ktab is (re)allocated             */
    /* submitters[]: aes_ctr_submit calls between their `running` check and their last slot store, counted per
     * thread shard: aes_engine_stop waits for all of them to reach 0 before it reads next_seq, so no sequence
     * number is published behind its back */
    /* every sequence number below this belongs to a run that has been stopped: complete, unless listed
     * in `lost` (requests an unclean stop -- dead kernel -- never saw complete)                        */
    std::atomic<uint64_t> done_upto{1};
    std::atomic<int> any_lost{0};
    std::mutex lost_mu;
    std::vector<uint64_t> lost;           /* sorted */
    bool broken = false;                  /* a CUDA call failed: rebuild everything at the next start */
};

/* One engine per GPU (requests shard over the GPUs of a node with no exchange
 * step); a handle carries its engine's device index in its top byte, the sequence number below.          */
Engine g_engs[AESOFF_MAX_DEVICES];
std::atomic<uint32_t> g_running_mask{0}; /* bit d: the engine on device d accepts requests                */
std::atomic<int> g_single{-1};           /* the device index if exactly one engine runs, else -1          */
std::atomic<uint32_t> g_round_robin{0};
std::mutex g_lifecycle;
constexpr int HANDLE_DEV_SHIFT = 56;
constexpr uint64_t HANDLE_SEQ_MASK = (1ull << HANDLE_DEV_SHIFT) - 1;

void publish_running(int device, bool on)
{
    uint32_t m = g_running_mask.load();
    m = on ? (m | (1u << device)) : (m & ~(1u << device));
    g_running_mask.store(m, std::memory_order_release);
    g_single.store(__builtin_popcount(m) == 1 ? __builtin_ctz(m) : -1, std::memory_order_release);
}

/* the owner of an address for the router: a device index, or AESOFF_OWNER_HOST */
int resolve_owner(const void *ptr)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, ptr) != cudaSuccess) {
        cudaGetLastError();
        return AESOFF_OWNER_HOST;
    }
    return a.type == cudaMemoryTypeDevice ? a.device : AESOFF_OWNER_HOST;
}

/* GPUs of the node (cudaGetDeviceCount at the last engine start) and the test hook AESOFF_ROUTE_ALWAYS=1, read at every
 * engine start: owners are looked up even where the answer cannot matter (one GPU, one engine), so that the look-up path
 * can be exercised against real CUDA addresses on a one-GPU box (tests/test_gpu_router.py).                            */
std::atomic<int> g_node_gpus{0};
std::atomic<int> g_route_always{0};

/* The engine a request goes to, or nullptr with *err = AES_E_STOPPED (none running / the GPU that owns its memory runs
 * none) or AES_E_INVAL (src and dst belong to two different GPUs: no engine can reach both -- peer access is never
 * enabled, include/aesoff.h).  Owners are not looked at only where there is nothing to decide and nothing to refuse: one
 * engine on a node with one GPU.  With one engine on a node with several GPUs the look-up stays (one remembered answer per
 * 2 MiB page and thread): memory of another GPU must be refused, not handed to a kernel that cannot address it.          */
Engine *route(const void *src, void *dst, size_t len, int *err)
{
    *err = AES_E_STOPPED;
    const int single = g_single.load(std::memory_order_acquire);
    if (single >= 0 && g_node_gpus.load(std::memory_order_relaxed) == 1 && !g_route_always.load(std::memory_order_relaxed))
        return &g_engs[single];
    const uint32_t mask = g_running_mask.load(std::memory_order_acquire);
    if (mask == 0) return nullptr;
    int so = AESOFF_OWNER_HOST, dO = AESOFF_OWNER_HOST;
    if (len) {
        dO = aesoff_route_owner_cached(dst, resolve_owner);
        so = src == dst ? dO : aesoff_route_owner_cached(src, resolve_owner);
    }
    uint32_t rr = g_round_robin.load(std::memory_order_relaxed);
    const int d = aesoff_route_decide(so, dO, mask, &rr);
    if (so < 0 && dO < 0) g_round_robin.store(rr, std::memory_order_relaxed);
    if (d == AESOFF_ROUTE_MIXED) *err = AES_E_INVAL;
    return d >= 0 ? &g_engs[d] : nullptr;
}
std::atomic<uint64_t> g_kernel_launches{0};

inline bool engine_dead(const Engine &e)
{
    return __atomic_load_n(&e.hctl[AESOFF_CTL_ALIVE], __ATOMIC_ACQUIRE) == 2u;
}

void free_engine_memory(Engine &e)
{
    /* key hygiene: raw keys sit in ring slots, expanded ones in ktab */
    if (e.hring) explicit_bzero(e.hring, (size_t)e.R * sizeof(aesoff_host_slot_t));
    if (e.ktab) cudaMemset(e.ktab, 0, (size_t)(AESOFF_KEY_IDS + e.R) * sizeof(aesoff_key_t));
    if (e.hring) cudaFreeHost(e.hring);
    if (e.hmail) cudaFreeHost(e.hmail);
    if (e.hctl) cudaFreeHost(e.hctl);
    if (e.dq) cudaFree(e.dq);
    if (e.tmap) cudaFree(e.tmap);
    if (e.ktab) cudaFree(e.ktab);
    if (e.counters) cudaFree(e.counters);
    if (e.dev_done_seq) cudaFree(e.dev_done_seq);
    if (e.dq_done) cudaFree(e.dq_done);
    if (e.dT0) cudaFree(e.dT0);
    if (e.stream) cudaStreamDestroy(e.stream);
    e.hring = nullptr;
    e.hmail = nullptr;
    e.hctl = nullptr;
    e.dq = nullptr;
    e.tmap = nullptr;
    e.ktab = nullptr;
    e.counters = e.dev_done_seq = nullptr;
    e.dq_done = e.dT0 = nullptr;
    e.stream = nullptr;
    {
        std::lock_guard<std::mutex> lk(e.id_mu);
        e.k_epoch.fetch_add(1);
        e.id_free.clear();
    }
}

void reset_key_ids(Engine &e)
{
    std::lock_guard<std::mutex> lk(e.id_mu);
    e.k_epoch.fetch_add(1);
    e.id_free.clear();
    for (uint32_t i = 0; i < AESOFF_KEY_IDS; ++i) e.id_free.emplace_back(i, 0ull);
}

/* a ktab index for a context, or AESOFF_KEY_NONE when none may be handed out right now */
uint32_t alloc_key_id(Engine &e)
{
    std::lock_guard<std::mutex> lk(e.id_mu);
    if (e.id_free.empty()) return AESOFF_KEY_NONE;
    const auto f = e.id_free.front();
    if (f.second != 0 && e.next_seq.load(std::memory_order_acquire) < f.second + e.R) return AESOFF_KEY_NONE;
    e.id_free.pop_front();
    return f.first;
}

inline bool is_pow2(uint32_t x) { return x && !(x & (x - 1)); }

/* geometry of a request, the same arithmetic the dispatcher warp does on the device */
inline void request_geometry(uint64_t len, uint8_t c0, uint32_t chunk_rows, uint32_t TM, uint64_t *rows,
                             uint32_t *crows, uint32_t *nchunks)
{
    const uint64_t nblocks = (len >> 4) + ((len & 15) ? 1 : 0);
    const uint64_t r = nblocks ? ((nblocks + c0 + AESOFF_ROW_BLOCKS - 1) >> 8) : 0;
    uint32_t cr = chunk_rows;
    const uint64_t max_chunks = TM / 4;
    while (((r + cr - 1) / cr) > max_chunks) cr *= 2;
    *rows = r;
    *crows = cr;
    *nchunks = (uint32_t)((r + cr - 1) / cr);
}

int check_buffers(const void *src, void *dst, size_t len)
{
    if (len == 0) return AES_OK;
    if (!src || !dst) return AES_E_INVAL;
    if ((uint64_t)len >= (1ull << 36)) return AES_E_INVAL; /* 64 GiB: the dispatcher counts 4 KiB rows in 32 bits */
    const uintptr_t s = (uintptr_t)src, d = (uintptr_t)dst;
    if ((s | d) & 15u) return AES_E_ALIGN;
    if (s != d && s < d + len && d < s + len) return AES_E_OVERLAP;
    return AES_OK;
}

} /* namespace */

/* ============================================================================================ */
/* errors                                                                                       */
/* ============================================================================================ */
extern "C" int aes_last_error(void) { return t_last_error; }

/* test hook (tests/test_gpu_restart.py): where a context's key stands on one engine, AESOFF_CTX_* */
extern "C" __attribute__((visibility("default"))) int aesoff_test_ctx_state(const aes_ctx_t *ctx, int device)
{
    if (!ctx || device < 0 || device >= AESOFF_MAX_DEVICES) return -1;
    return (int)__atomic_load_n(&ctx->dev[device].state, __ATOMIC_ACQUIRE);
}

/* for aes_ctr_launch_static, which lives beside its static array in aesoff_kernels.cu */
extern "C" int aesoff_fail(int code) { return fail(code); }
extern "C" void aesoff_note_launches(int n) { g_kernel_launches.fetch_add((uint64_t)n); }

extern "C" const char *aes_strerror(int code)
{
    switch (code) {
    case AES_OK: return "ok";
    case AES_E_INVAL: return "invalid argument";
    case AES_E_KEYBITS: return "keybits must be 128, 192 or 256";
    case AES_E_ALIGN: return "src/dst must be 16-byte aligned";
    case AES_E_OVERLAP: return "src and dst overlap partially";
    case AES_E_AGAIN: return "submission ring full";
    case AES_E_TIMEOUT: return "timed out";
    case AES_E_STOPPED: return "engine not running";
    case AES_E_CUDA: return "CUDA error or no device";
    case AES_E_BUSY: return "not allowed while the engine is running";
    case AES_E_NOMEM: return "out of memory";
    case AES_E_TOOBIG: return "request larger than AES_STATIC_MAX_BYTES (aes_ctr_launch_static has no memory to grow into)";
    default: return "unknown error";
    }
}

/* ============================================================================================ */
/* contexts (step a1)                                                                           */
/* ============================================================================================ */
extern "C" aes_ctx_t *aes_ctx_create(const uint8_t *key, int keybits)
{
    if (!key) {
        fail(AES_E_INVAL);
        return nullptr;
    }
    if (keybits != 128 && keybits != 192 && keybits != 256) {
        fail(AES_E_KEYBITS);
        return nullptr;
    }
    aes_ctx_t *c = (aes_ctx_t *)malloc(sizeof(aes_ctx_t));
    if (!c) {
        fail(AES_E_NOMEM);
        return nullptr;
    }
    /* the host expansion (aesoff_keys.cpp) is done on demand: the engine path ships the raw key and the
     * dispatcher warp expands it, so a per-request context (BASELINE.json configs[3]) never pays for it */
    c->nr = keybits / 32 + 6;
    c->rk_ready = 0;
    c->keybits = keybits;
    memset(c->key, 0, sizeof(c->key));
    for (int i = 0; i < keybits / 32; ++i)
        c->key[i] = (uint32_t)key[4 * i] | ((uint32_t)key[4 * i + 1] << 8) | ((uint32_t)key[4 * i + 2] << 16) |
                    ((uint32_t)key[4 * i + 3] << 24);
    for (int d = 0; d < AESOFF_MAX_DEVICES; ++d) {
        c->dev[d].state = AESOFF_CTX_FRESH;
        c->dev[d].id = AESOFF_KEY_NONE;
        c->dev[d].epoch = 0;
        c->dev[d].install_seq = 0;
    }
    return c;
}

extern "C" void aes_ctx_destroy(aes_ctx_t *ctx)
{
    if (!ctx) return;
    for (int d = 0; d < AESOFF_MAX_DEVICES; ++d) {
        aes_ctx_dev &k = ctx->dev[d];
        if (__atomic_load_n(&k.state, __ATOMIC_ACQUIRE) >= AESOFF_CTX_INSTALLING && k.id != AESOFF_KEY_NONE) {
            Engine &e = g_engs[d];
            std::lock_guard<std::mutex> lk(e.id_mu);
            /* requests in flight may still name the index: it rests until they must have completed */
            if (k.epoch == e.k_epoch.load()) e.id_free.emplace_back(k.id, e.next_seq.load());
        }
    }
    explicit_bzero(ctx, sizeof(*ctx)); /* key hygiene: raw key and round keys do not outlive the context */
    free(ctx);
}

namespace {
std::mutex g_rk_mu;
/* fills ctx->rk from ctx->key once (thread-safe) */
void host_round_keys(aes_ctx_t *ctx)
{
    if (__atomic_load_n(&ctx->rk_ready, __ATOMIC_ACQUIRE)) return;
    std::lock_guard<std::mutex> lk(g_rk_mu);
    if (ctx->rk_ready) return;
    uint8_t key[32];
    for (int i = 0; i < 8; ++i) {
        key[4 * i + 0] = (uint8_t)(ctx->key[i]);
        key[4 * i + 1] = (uint8_t)(ctx->key[i] >> 8);
        key[4 * i + 2] = (uint8_t)(ctx->key[i] >> 16);
        key[4 * i + 3] = (uint8_t)(ctx->key[i] >> 24);
    }
    aesoff_key_expand(key, ctx->keybits, ctx->rk);
    __atomic_store_n(&ctx->rk_ready, 1u, __ATOMIC_RELEASE);
}
} /* namespace */

extern "C" int aes_ctx_round_keys(const aes_ctx_t *ctx_in, uint8_t *out)
{
    if (!ctx_in || !out) return fail(AES_E_INVAL);
    aes_ctx_t *ctx = const_cast<aes_ctx_t *>(ctx_in);
    host_round_keys(ctx);
    /* little-endian words back to the FIPS-197 byte string */
    for (int i = 0; i < 4 * (ctx->nr + 1); ++i) {
        out[4 * i + 0] = (uint8_t)(ctx->rk[i]);
        out[4 * i + 1] = (uint8_t)(ctx->rk[i] >> 8);
        out[4 * i + 2] = (uint8_t)(ctx->rk[i] >> 16);
        out[4 * i + 3] = (uint8_t)(ctx->rk[i] >> 24);
    }
    return ctx->nr;
}

/* ============================================================================================ */
/* engine life cycle (step a0)                                                                  */
/* ============================================================================================ */
extern "C" int aes_engine_start(int device, const aes_engine_opts_t *opts)
{
    std::lock_guard<std::mutex> lk(g_lifecycle);
    if (device < 0 || device >= AESOFF_MAX_DEVICES) return fail(AES_E_CUDA);
    Engine &e = g_engs[device];
    if (e.running.load()) return fail(AES_E_BUSY);

    aes_engine_opts_t o;
    memset(&o, 0, sizeof(o));
    if (opts) o = *opts;
    if (o.reserved[0] || (o.flags & ~AES_ENGINE_NO_DECRYPT)) return fail(AES_E_INVAL);
    if (o.n_dispatchers == 0) o.n_dispatchers = AESOFF_DEF_DISPATCHERS;
    if (o.n_dispatchers > AESOFF_MAX_DISPATCHERS) return fail(AES_E_INVAL);
    if (o.ring_slots == 0) o.ring_slots = 2048;
    if (o.chunk_rows == 0) o.chunk_rows = 4;
    if (!is_pow2(o.ring_slots) || o.ring_slots < 64 || o.ring_slots > 4096) return fail(AES_E_INVAL);
    if (o.chunk_rows > 64 || !is_pow2(o.chunk_rows)) return fail(AES_E_INVAL);
    if (o.fine_rows == 0) o.fine_rows = 0xfffffffeu;
    if (o.fine_rows == AES_FINE_ROWS_OFF) o.fine_rows = 0;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return fail(AES_E_CUDA);
    g_node_gpus.store(ndev, std::memory_order_relaxed);
    {
        const char *ra = getenv("AESOFF_ROUTE_ALWAYS");
        g_route_always.store(ra && ra[0] == '1', std::memory_order_relaxed);
    }
    AesoffDeviceScope on_device(device); /* the caller's current device is restored on every return below */
    if (!on_device.ok) return fail(AES_E_CUDA);
    int sms = 0, major = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device);
    if (major != 10) return fail(AES_E_CUDA); /* sm_100a code only */

    /* ring, mailbox and queues survive a stop/start cycle with the same geometry (a restart then costs
     * one launch, not a dozen allocations) */
    const bool reuse = e.hring && !e.broken && e.device == device && e.R == o.ring_slots;
    e.broken = false;
    if (!reuse) free_engine_memory(e);
    e.device = device;
    e.sm_count = sms;
    e.n_ctas = o.n_ctas ? (int)o.n_ctas : sms;
    e.n_disp = o.n_dispatchers < (uint32_t)e.n_ctas ? o.n_dispatchers : (uint32_t)e.n_ctas;
    e.R = o.ring_slots;
    e.Rm = e.R - 1;
    e.chunk_rows = o.chunk_rows;
    e.TM = 1u << 18;
    e.first_seq = e.next_seq.load();

    bool ok = true;
    if (!reuse) {
    ok = ok && cudaStreamCreateWithFlags(&e.stream, cudaStreamNonBlocking) == cudaSuccess;
    const unsigned hflags = cudaHostAllocMapped | cudaHostAllocPortable;
    ok = ok && cudaHostAlloc((void **)&e.hring, (size_t)e.R * sizeof(aesoff_host_slot_t), hflags) == cudaSuccess;
    ok = ok && cudaHostAlloc((void **)&e.hmail, (size_t)e.R * 8, hflags) == cudaSuccess;
    ok = ok && cudaHostAlloc((void **)&e.hctl, AESOFF_CTL_WORDS * 4, hflags) == cudaSuccess;
    ok = ok && cudaMalloc((void **)&e.dq, (size_t)e.R * sizeof(aesoff_dq_entry_t)) == cudaSuccess;
    ok = ok && cudaMalloc((void **)&e.tmap, (size_t)e.TM * sizeof(aesoff_ticket_t)) == cudaSuccess;
    ok = ok && cudaMalloc((void **)&e.ktab, (size_t)(AESOFF_KEY_IDS + e.R) * sizeof(aesoff_key_t)) == cudaSuccess;
    ok = ok && cudaMalloc((void **)&e.counters, AESOFF_CNT_WORDS * 8) == cudaSuccess;
    ok = ok && cudaMalloc((void **)&e.dev_done_seq, (size_t)e.R * 8) == cudaSuccess;
    ok = ok && cudaMalloc((void **)&e.dq_done, (size_t)e.R * 4) == cudaSuccess;
    ok = ok && cudaMalloc((void **)&e.dT0, 512 * 4) == cudaSuccess;
    if (!ok) {
        free_engine_memory(e);
        return fail(AES_E_NOMEM);
    }
    memset(e.hring, 0, (size_t)e.R * sizeof(aesoff_host_slot_t));
    memset(e.hmail, 0, (size_t)e.R * 8);
    ok = ok && cudaMemset(e.dev_done_seq, 0, (size_t)e.R * 8) == cudaSuccess;
    ok = ok && cudaMemset(e.dq, 0, (size_t)e.R * sizeof(aesoff_dq_entry_t)) == cudaSuccess; /* no tag matches yet */
    ok = ok && cudaMemcpy(e.dT0, aesoff_T0_table(), 512 * 4, cudaMemcpyHostToDevice) == cudaSuccess;
    if (ok) reset_key_ids(e);
    }
    /* sequence numbers never restart, so stale slot/mailbox values (< first_seq) can never match */
    memset(e.hctl, 0, AESOFF_CTL_WORDS * 4);
    ok = ok && cudaMemsetAsync(e.counters, 0, AESOFF_CNT_WORDS * 8, e.stream) == cudaSuccess;
    /* the dispatchers' token: no ticket published yet, the first request to dispatch is first_seq */
    const uint64_t chain0[2] = {0ull, e.first_seq};
    ok = ok && cudaMemcpyAsync(e.counters + AESOFF_CNT_CHAIN, chain0, 16, cudaMemcpyHostToDevice, e.stream) == cudaSuccess;
    ok = ok && cudaMemsetAsync(e.dq_done, 0, (size_t)e.R * 4, e.stream) == cudaSuccess;
    /* ticket numbers restart from 0 with every launch: no stale ticket may carry a matching tag */
    ok = ok && cudaMemsetAsync(e.tmap, 0, (size_t)e.TM * sizeof(aesoff_ticket_t), e.stream) == cudaSuccess;
    if (!ok) {
        free_engine_memory(e);
        return fail(AES_E_CUDA);
    }

    aesoff_params_t p;
    memset(&p, 0, sizeof(p));
    p.hring = e.hring;
    p.hmail = e.hmail;
    p.hctl = e.hctl;
    p.dq = e.dq;
    p.ktab = e.ktab;
    p.tmap = e.tmap;
    p.counters = e.counters;
    p.dq_done = e.dq_done;
    p.dev_done_seq = e.dev_done_seq;
    p.T0 = e.dT0;
    p.R = e.R;
    p.TM = e.TM;
    p.chunk_rows = e.chunk_rows;
    for (p.chunk_log2 = 0; (1u << p.chunk_log2) < e.chunk_rows; ++p.chunk_log2) {}
    p.mode = AESOFF_MODE_PERSISTENT;
    p.idle_exit_ms = o.idle_exit_ms;
    p.fine_rows = o.fine_rows;
    p.first_seq = e.first_seq;
    p.n_disp = e.n_disp;
    p.need_dec = (o.flags & AES_ENGINE_NO_DECRYPT) ? 0u : 1u;
    e.has_dec = p.need_dec != 0;
    {   /* unit-size policy thresholds in rows (aesoff_shared.h AESOFF_TUNE_*); W = worker warps of the grid.
         * AESOFF_TUNE="a,b,c,d,e,f,g" overrides them (tuning experiments only). */
        const uint32_t W = (uint32_t)e.n_ctas * AESOFF_WORKER_WARPS;
        p.tune[AESOFF_TUNE_FINE_TOTAL] = W / 4;
        p.tune[AESOFF_TUNE_FINE_FRONT] = 0;
        p.tune[AESOFF_TUNE_HALF_TOTAL] = 3 * W / 4;
        p.tune[AESOFF_TUNE_TAIL_AHEAD] = W;
        p.tune[AESOFF_TUNE_TAIL_LEFT] = 2 * W;
        p.tune[AESOFF_TUNE_SPREAD_AHEAD] = W / 2;
        p.tune[AESOFF_TUNE_SPREAD_MAX] = 16;
        p.tune[AESOFF_TUNE_POLL_DEPTH] = 3;
        p.tune[AESOFF_TUNE_POLL_GAP] = 350;
        p.tune[AESOFF_TUNE_PRERESERVE] = 4;
        if (const char *t = getenv("AESOFF_TUNE")) {
            for (int i = 0; i < 10 && t && *t; ++i) {
                char *end = nullptr;
                const unsigned long v = strtoul(t, &end, 10);
                if (end != t) p.tune[i] = (uint32_t)v;
                t = (*end == ',') ? end + 1 : nullptr;
            }
            if (p.tune[AESOFF_TUNE_POLL_DEPTH] < 1u) p.tune[AESOFF_TUNE_POLL_DEPTH] = 1u;
            if (p.tune[AESOFF_TUNE_POLL_DEPTH] > 3u) p.tune[AESOFF_TUNE_POLL_DEPTH] = 3u;
        }
    }
    if (aesoff_launch_engine(&p, e.n_ctas, e.stream) != 0) {
        free_engine_memory(e);
        return fail(AES_E_CUDA);
    }
    g_kernel_launches.fetch_add(1);
    /* wait until the dispatcher warp is really polling (bounded) */
    const uint64_t t0 = now_ns();
    while (__atomic_load_n(&e.hctl[AESOFF_CTL_ALIVE], __ATOMIC_ACQUIRE) == 0u) {
        if (now_ns() - t0 > 20ull * 1000000000ull || cudaStreamQuery(e.stream) != cudaErrorNotReady) {
            /* A kernel that was only waiting for the SMs may still start: it must find STOP in memory that is still
             * mapped, so the stream is waited for (the kernel sees STOP and leaves, or has failed) before anything
             * is freed.                                                                                            */
            __atomic_store_n(&e.hctl[AESOFF_CTL_STOP], 1u, __ATOMIC_RELEASE);
            cudaStreamSynchronize(e.stream);
            cudaGetLastError();
            free_engine_memory(e);
            return fail(AES_E_CUDA);
        }
        CPU_RELAX();
    }
    if (engine_dead(e)) {
        /* The kernel has already come and gone (ALIVE == 2): the launch was serialised -- a profiler, a
         * sanitizer or CUDA_LAUNCH_BLOCKING makes the launch call wait for the kernel, which then sits out
         * its idle timer with nobody able to submit.  A dead engine is not a running one.               */
        cudaStreamSynchronize(e.stream);
        return fail(AES_E_STOPPED);
    }
    e.running.store(1, std::memory_order_release);
    publish_running(device, true);
    return AES_OK;
}

namespace {
/* g_lifecycle held */
int stop_engine(Engine &e)
{
    if (!e.running.load()) return fail(AES_E_STOPPED);
    /* no new submissions from here on; the ones that passed their `running` check finish publishing */
    publish_running(e.device, false);
    e.running.store(2, std::memory_order_seq_cst);
    for (int i = 0; i < SUBMIT_SHARDS; ++i)
        while (e.submitters[i].n.load(std::memory_order_seq_cst) != 0) CPU_RELAX();
    int rc = AES_OK;
    /* drain: every accepted request completes (unless the kernel died) */
    const uint64_t last = e.next_seq.load();
    const uint64_t lo = (last > e.first_seq + e.R) ? last - e.R : e.first_seq;
    for (uint64_t s = lo; s < last; ++s) {
        const uint64_t t0 = now_ns();
        while (__atomic_load_n(&e.hmail[(s - 1) & e.Rm], __ATOMIC_ACQUIRE) < s) {
            if (engine_dead(e) || now_ns() - t0 > 60ull * 1000000000ull) {
                rc = AES_E_STOPPED;
                break;
            }
            CPU_RELAX();
        }
        if (rc != AES_OK) break;
    }
    __atomic_store_n(&e.hctl[AESOFF_CTL_STOP], 1u, __ATOMIC_RELEASE);
    if (cudaStreamSynchronize(e.stream) != cudaSuccess) rc = AES_E_CUDA;
    if (rc != AES_OK) {
        /* unclean stop: the requests the mailbox never saw complete are lost, and aes_poll says so */
        std::lock_guard<std::mutex> ll(e.lost_mu);
        for (uint64_t s = lo; s < last; ++s)
            if (__atomic_load_n(&e.hmail[(s - 1) & e.Rm], __ATOMIC_ACQUIRE) < s) e.lost.push_back(s);
        if (e.lost.size() > 65536) e.lost.erase(e.lost.begin(), e.lost.end() - 65536);
        e.any_lost.store(e.lost.empty() ? 0 : 1, std::memory_order_release);
        /* a lost request may be one that was to file a key in ktab: every installed context installs again */
        reset_key_ids(e);
    }
    e.done_upto.store(last, std::memory_order_release);
    /* ring, mailbox and queues are kept for the next start (aes_poll may still be reading the mailbox);
     * after a CUDA error the next start rebuilds them */
    if (rc == AES_E_CUDA) e.broken = true;
    e.running.store(0, std::memory_order_release);
    if (rc != AES_OK) return fail(rc);
    return AES_OK;
}
} /* namespace */

extern "C" int aes_engine_stop_device(int device)
{
    std::lock_guard<std::mutex> lk(g_lifecycle);
    if (device < 0 || device >= AESOFF_MAX_DEVICES) return fail(AES_E_INVAL);
    return stop_engine(g_engs[device]);
}

extern "C" int aes_engine_stop(void)
{
    std::lock_guard<std::mutex> lk(g_lifecycle);
    int rc = AES_E_STOPPED, n = 0;
    for (int d = 0; d < AESOFF_MAX_DEVICES; ++d)
        if (g_engs[d].running.load()) {
            const int r = stop_engine(g_engs[d]);
            if (n++ == 0 || r != AES_OK) rc = r;
        }
    if (rc != AES_OK) return fail(rc);
    return AES_OK;
}

extern "C" int aes_engine_info_device(int device, aes_engine_info_t *out)
{
    if (!out || device < 0 || device >= AESOFF_MAX_DEVICES) return fail(AES_E_INVAL);
    memset(out, 0, sizeof(*out));
    Engine &e = g_engs[device];
    out->engines_running = (uint32_t)__builtin_popcount(g_running_mask.load());
    out->running = e.running.load() == 1 && e.hctl && !engine_dead(e);
    out->device = e.device;
    out->sm_count = e.sm_count;
    out->n_ctas = e.n_ctas;
    out->threads_per_cta = AESOFF_CTA_THREADS;
    out->worker_warps_per_cta = AESOFF_WORKER_WARPS;
    out->ring_slots = e.R;
    out->chunk_rows = e.chunk_rows;
    out->smem_bytes_per_cta = e.has_dec ? AESOFF_SMEM_BYTES : AESOFF_SMEM_BYTES_NODEC;
    const uint64_t next = e.next_seq.load();
    out->submitted = next - 1;
    uint64_t pending = 0;
    if (e.running.load() && e.hmail) {
        for (uint64_t s = (next > e.first_seq + e.R) ? next - e.R : e.first_seq; s < next; ++s)
            if (__atomic_load_n(&e.hmail[(s - 1) & e.Rm], __ATOMIC_ACQUIRE) < s) ++pending;
    }
    out->completed = out->submitted - pending;
    out->kernel_launches = g_kernel_launches.load();
    out->n_dispatchers = e.n_disp;
    if (e.hctl) {
        for (uint32_t d = 0; d < AESOFF_MAX_DISPATCHERS; ++d) { /* one set per dispatcher warp */
            const uint32_t *st = e.hctl + AESOFF_CTL_STATS + AESOFF_CTL_STAT_WORDS * d;
            out->cut_eighths += __atomic_load_n(&st[AESOFF_CTL_CUT_EIGHTHS], __ATOMIC_RELAXED);
            out->cut_halves += __atomic_load_n(&st[AESOFF_CTL_CUT_HALVES], __ATOMIC_RELAXED);
            out->cut_rows += __atomic_load_n(&st[AESOFF_CTL_CUT_ROWS], __ATOMIC_RELAXED);
        }
    }
    return AES_OK;
}

/* the running engine on the lowest device; if none runs, the one that ran last on the lowest device */
extern "C" int aes_engine_info(aes_engine_info_t *out)
{
    int pick = 0;
    const uint32_t m = g_running_mask.load();
    if (m) {
        pick = __builtin_ctz(m);
    } else {
        for (int d = 0; d < AESOFF_MAX_DEVICES; ++d)
            if (g_engs[d].device >= 0) {
                pick = d;
                break;
            }
    }
    return aes_engine_info_device(pick, out);
}

/* -DAESOFF_WSTATS builds: {clocks inside units, clocks waiting between units, units} summed over all worker warps of the
 * engine run that was stopped last on `device` (read after aes_engine_stop); zeros otherwise.  Tuning aid, not in aesoff.h. */
extern "C" __attribute__((visibility("default"))) int aesoff_debug_worker_stats(int device, uint64_t out[3])
{
    if (device < 0 || device >= AESOFF_MAX_DEVICES || !g_engs[device].counters) return -1;
    return cudaMemcpy(out, g_engs[device].counters + AESOFF_CNT_DEBUG, 24, cudaMemcpyDeviceToHost) == cudaSuccess ? 0 : -1;
}

/* AESOFF_DISP_STATS builds: per-dispatcher counters (polls that took requests, requests, token wait and work
 * in units of 64 ns, empty polls), 5 words per dispatcher; zeros otherwise.  Tuning aid, not in aesoff.h.   */
extern "C" __attribute__((visibility("default"))) int aesoff_debug_dispatch_stats(uint32_t out[5 * AESOFF_MAX_DISPATCHERS])
{
    Engine &e = g_engs[g_single.load() >= 0 ? g_single.load() : 0];
    if (!e.hctl) return -1;
    for (uint32_t d = 0; d < AESOFF_MAX_DISPATCHERS; ++d)
        for (int i = 0; i < 5; ++i)
            out[5 * d + i] = __atomic_load_n(&e.hctl[AESOFF_CTL_STATS + AESOFF_CTL_STAT_WORDS * d + AESOFF_CTL_DBG_TAKES + i], __ATOMIC_RELAXED);
    return 0;
}

/* ============================================================================================ */
/* submit / poll / wait (steps a2, a7)                                                          */
/* ============================================================================================ */
namespace {
/* mode: AESOFF_MODE_*; nonce: the ICB (CTR), the IV (CBC) or 16 zero bytes (ECB) */
aes_handle_t submit_mode(aes_ctx_t *ctx, uint32_t mode, const uint8_t nonce[16], const void *src, void *dst, size_t len)
{
    if (!ctx || !nonce) {
        fail(AES_E_INVAL);
        return 0;
    }
    int rc = check_buffers(src, dst, len);
    if (rc == AES_OK && mode != AESOFF_MODE_CTR && (len & 15u)) rc = AES_E_INVAL;             /* whole blocks only */
    if (rc == AES_OK && mode == AESOFF_MODE_CBC_DEC && len && src == dst) rc = AES_E_OVERLAP; /* see aesoff.h */
    if (rc != AES_OK) {
        fail(rc);
        return 0;
    }
    int route_err = AES_E_STOPPED;
    Engine *ep = route(src, dst, len, &route_err);
    if (!ep) {
        fail(route_err);
        return 0;
    }
    Engine &e = *ep;
    if ((mode == AESOFF_MODE_ECB_DEC || mode == AESOFF_MODE_CBC_DEC) && !e.has_dec) {
        fail(AES_E_INVAL); /* started with AES_ENGINE_NO_DECRYPT */
        return 0;
    }
    aes_ctx_dev &ck = ctx->dev[e.device];
    /* counted BEFORE the running check: aes_engine_stop sets running = 2 and then waits for the count to
     * drop to 0, so a submit either fails here or has published its slot before the drain reads next_seq */
    struct InFlight {
        std::atomic<int> &n;
        explicit InFlight(std::atomic<int> &c) : n(c) { n.fetch_add(1, std::memory_order_seq_cst); }
        ~InFlight() { n.fetch_sub(1, std::memory_order_seq_cst); }
    } in_flight(e.submitters[thread_shard()].n);
    if (e.running.load(std::memory_order_seq_cst) != 1 || engine_dead(e)) {
        fail(AES_E_STOPPED);
        return 0;
    }
    /* how the key travels (aesoff_internal.h): raw until the request that files the expanded key in ktab
     * has completed, by ktab index afterwards.  Completion is what orders the two: the dispatcher warps take
     * batches of requests side by side, so a lower sequence number alone does not mean "expanded first". */
    uint32_t kw = ((uint32_t)ctx->nr << 24) | AESOFF_KEY_NONE | AESOFF_KW_RAW;
    bool installing = false;
    /* state and epoch are two words: read the state again after the epoch and start over if another thread moved it in
     * between (a re-install after a rebuilt key table goes INSTALLED/INSTALLING -> CLAIMED -> INSTALLING with the NEW epoch;
     * a stale INSTALLED paired with the new epoch would name a table entry that has not been filled yet)               */
    uint32_t st;
    uint64_t epoch_now;
    bool epoch_ok;
    do {
        st = __atomic_load_n(&ck.state, __ATOMIC_ACQUIRE);
        epoch_now = e.k_epoch.load(std::memory_order_acquire);
        epoch_ok = __atomic_load_n(&ck.epoch, __ATOMIC_ACQUIRE) == epoch_now;
    } while (__atomic_load_n(&ck.state, __ATOMIC_ACQUIRE) != st);
    if (st == AESOFF_CTX_INSTALLING && epoch_ok) {
        const uint64_t is = __atomic_load_n(&ck.install_seq, __ATOMIC_ACQUIRE);
        if (is != 0 && __atomic_load_n(&e.hmail[(is - 1) & e.Rm], __ATOMIC_ACQUIRE) >= is) {
            __atomic_store_n(&ck.state, AESOFF_CTX_INSTALLED, __ATOMIC_RELEASE);
            st = AESOFF_CTX_INSTALLED;
        }
    }
    if (st == AESOFF_CTX_INSTALLED && epoch_ok) {
        kw = ((uint32_t)ctx->nr << 24) | ck.id;
    } else if (st == AESOFF_CTX_FRESH) {
        __atomic_compare_exchange_n(&ck.state, &st, AESOFF_CTX_SEEN, false, __ATOMIC_ACQ_REL, __ATOMIC_ACQUIRE);
    } else if (st == AESOFF_CTX_SEEN || ((st == AESOFF_CTX_INSTALLED || st == AESOFF_CTX_INSTALLING) && !epoch_ok)) {
        /* INSTALLED, or INSTALLING with nobody having looked at the install's completion yet, under an older ktab
         * generation (the engine was rebuilt, or stopped uncleanly): install again.  The winner holds the entry in
         * CLAIMED while it fills id, epoch and install_seq, so INSTALLING always comes with a consistent triple.    */
        const uint32_t id = alloc_key_id(e);
        if (id != AESOFF_KEY_NONE) {
            if (__atomic_compare_exchange_n(&ck.state, &st, AESOFF_CTX_CLAIMED, false, __ATOMIC_ACQ_REL,
                                            __ATOMIC_ACQUIRE)) {
                __atomic_store_n(&ck.install_seq, 0ull, __ATOMIC_RELEASE);
                ck.id = id;
                __atomic_store_n(&ck.epoch, epoch_now, __ATOMIC_RELEASE);
                __atomic_store_n(&ck.state, AESOFF_CTX_INSTALLING, __ATOMIC_RELEASE);
                kw |= AESOFF_KW_INSTALL;
                kw = (kw & ~0xffffu) | id;
                installing = true;
            } else {
                std::lock_guard<std::mutex> lk(e.id_mu); /* another thread got there first */
                e.id_free.emplace_front(id, 0ull);
            }
        }
    } /* else: INSTALLING and not complete yet, or CLAIMED (another thread is in the middle of it): raw, nothing stored */
    /* claim the next sequence number, but only if its slot has been vacated */
    uint64_t s = e.next_seq.load(std::memory_order_acquire);
    for (;;) {
        if (s - e.first_seq >= e.R &&
            __atomic_load_n(&e.hmail[(s - 1) & e.Rm], __ATOMIC_ACQUIRE) < s - e.R) {
            if (installing) { /* undo: the index was never named by a descriptor */
                {
                    std::lock_guard<std::mutex> lk(e.id_mu);
                    e.id_free.emplace_front(ck.id, 0ull);
                }
                ck.id = AESOFF_KEY_NONE;
                __atomic_store_n(&ck.epoch, 0ull, __ATOMIC_RELEASE);
                __atomic_store_n(&ck.state, AESOFF_CTX_SEEN, __ATOMIC_RELEASE);
            }
            fail(AES_E_AGAIN);
            return 0;
        }
        if (e.next_seq.compare_exchange_weak(s, s + 1, std::memory_order_acq_rel)) break;
    }
    const uint32_t tag = (uint32_t)s;
    const uint64_t a_src = (uint64_t)(uintptr_t)src, a_dst = (uint64_t)(uintptr_t)dst, a_len = (uint64_t)len;
    uint32_t icb[4];
    memcpy(icb, nonce, 16);
    uint32_t *w = e.hring[(s - 1) & e.Rm].w;
    /* second line first: the dispatcher wants it whenever line one says RAW.  It is rewritten by EVERY
     * submit (zeros when the key travels by index): tags are the low 32 bits of the sequence number, and a
     * raw-key line left over from 2^32 requests ago must never be paired with a fresh first line.        */
    if (kw & AESOFF_KW_RAW) {
        store_piece(w + 16, ctx->key[0], ctx->key[1], ctx->key[2], tag);
        store_piece(w + 20, ctx->key[3], ctx->key[4], ctx->key[5], tag);
        store_piece(w + 24, ctx->key[6], ctx->key[7], 0u, tag);
        store_piece(w + 28, 0u, 0u, 0u, tag);
    } else {
        store_piece(w + 16, 0u, 0u, 0u, tag);
        store_piece(w + 20, 0u, 0u, 0u, tag);
        store_piece(w + 24, 0u, 0u, 0u, tag);
        store_piece(w + 28, 0u, 0u, 0u, tag);
    }
    store_piece(w + 0, icb[0], icb[1], icb[2], tag);
    store_piece(w + 4, icb[3], (uint32_t)a_src, (uint32_t)(a_src >> 32), tag);
    store_piece(w + 8, (uint32_t)a_dst, (uint32_t)(a_dst >> 32), (uint32_t)a_len, tag);
    store_piece(w + 12, (uint32_t)(a_len >> 32), kw, mode, tag);
    /* later submits name ktab[id] once this request, which fills it, has completed */
    if (installing) __atomic_store_n(&ck.install_seq, s, __ATOMIC_RELEASE);
    return (aes_handle_t)(s | ((uint64_t)e.device << HANDLE_DEV_SHIFT));
}
const uint8_t k_zero_iv[16] = {0};
} /* namespace */

extern "C" aes_handle_t aes_ctr_submit(aes_ctx_t *ctx, const uint8_t nonce[16], const void *src, void *dst, size_t len)
{
    return submit_mode(ctx, AESOFF_MODE_CTR, nonce, src, dst, len);
}
extern "C" aes_handle_t aes_ecb_submit(aes_ctx_t *ctx, int decrypt, const void *src, void *dst, size_t len)
{
    return submit_mode(ctx, decrypt ? AESOFF_MODE_ECB_DEC : AESOFF_MODE_ECB_ENC, k_zero_iv, src, dst, len);
}
extern "C" aes_handle_t aes_cbc_decrypt_submit(aes_ctx_t *ctx, const uint8_t iv[16], const void *src, void *dst, size_t len)
{
    return submit_mode(ctx, AESOFF_MODE_CBC_DEC, iv, src, dst, len);
}

extern "C" int aes_poll(aes_handle_t h)
{
    /* A valid handle is below its engine's next_seq.  That word is claimed by every submit of every thread, so a
     * poll does not read it: it compares with this thread's last copy and refreshes the copy only for a handle above it. */
    thread_local uint64_t seen_next[AESOFF_MAX_DEVICES] = {0};
    const unsigned dev = (unsigned)(h >> HANDLE_DEV_SHIFT);
    if (dev >= AESOFF_MAX_DEVICES) return fail(AES_E_INVAL);
    Engine &e = g_engs[dev];
    h &= HANDLE_SEQ_MASK;
    if (h == 0) return fail(AES_E_INVAL);
    if (h >= seen_next[dev]) {
        seen_next[dev] = e.next_seq.load(std::memory_order_acquire);
        if (h >= seen_next[dev]) return fail(AES_E_INVAL);
    }
    if (h < e.done_upto.load(std::memory_order_acquire)) {
        /* a run that has been stopped: a clean stop drained everything, an unclean one lists what it lost */
        if (e.any_lost.load(std::memory_order_acquire)) {
            std::lock_guard<std::mutex> lk(e.lost_mu);
            if (std::binary_search(e.lost.begin(), e.lost.end(), (uint64_t)h)) return fail(AES_E_STOPPED);
        }
        return 1;
    }
    if (!e.hmail) return fail(AES_E_STOPPED);
    if (__atomic_load_n(&e.hmail[(h - 1) & e.Rm], __ATOMIC_ACQUIRE) >= h) return 1;
    if (engine_dead(e)) {
        /* the exit path of the kernel cannot overtake a completion it already signalled */
        if (__atomic_load_n(&e.hmail[(h - 1) & e.Rm], __ATOMIC_ACQUIRE) >= h) return 1;
        return fail(AES_E_STOPPED);
    }
    return 0;
}

/* Spins (pause) for the first ~20 us -- the offloads this engine is built for complete in 10 -- then yields the
 * core between polls, then sleeps in growing steps up to 50 us: a 32-thread executor waiting on
 * long requests does not burn 32 cores.                                                                       */
extern "C" int aes_wait(aes_handle_t h, uint64_t timeout_ns)
{
    const uint64_t t0 = now_ns();
    uint32_t sleep_ns = 1000;
    for (uint32_t spins = 0;; ++spins) {
        const int r = aes_poll(h);
        if (r == 1) return AES_OK;
        if (r < 0) return r;
        if (spins < 2048u) {
            if ((spins & 63u) == 63u && timeout_ns != UINT64_MAX && now_ns() - t0 > timeout_ns) return fail(AES_E_TIMEOUT);
            CPU_RELAX();
            continue;
        }
        if (timeout_ns != UINT64_MAX && now_ns() - t0 > timeout_ns) return fail(AES_E_TIMEOUT);
        if (spins < 2048u + 256u) {
            sched_yield();
        } else {
            struct timespec ts = {0, (long)sleep_ns};
            nanosleep(&ts, nullptr);
            if (sleep_ns < 50000u) sleep_ns *= 2;
        }
    }
}

extern "C" void aes_route_flush(void) { aesoff_route_flush_cache(); }

/* ============================================================================================ */
/* pinned host memory                                                                            */
/* ============================================================================================ */
extern "C" void *aes_host_alloc(size_t bytes)
{
    void *p = nullptr;
    if (cudaHostAlloc(&p, bytes ? bytes : 1, cudaHostAllocMapped | cudaHostAllocPortable) != cudaSuccess) {
        cudaGetLastError();
        fail(AES_E_CUDA);
        return nullptr;
    }
    return p;
}
extern "C" void aes_host_free(void *p)
{
    if (p) cudaFreeHost(p);
}

/* A buffer the server already owns (malloc, a slab, a network buffer: the paper's j.buf): page-lock it
 * where it lies and make it GPU-addressable, so that it can be submitted as it is.                              */
extern "C" int aes_host_register(void *ptr, size_t bytes)
{
    if (!ptr || bytes == 0) return fail(AES_E_INVAL);
    const cudaError_t e = cudaHostRegister(ptr, bytes, cudaHostRegisterMapped | cudaHostRegisterPortable);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(e == cudaErrorMemoryAllocation ? AES_E_NOMEM : e == cudaErrorInvalidValue ? AES_E_INVAL : AES_E_CUDA);
    }
    void *dp = nullptr;
    /* with unified addressing the device sees registered memory at its host address; the kernel uses that address */
    if (cudaHostGetDevicePointer(&dp, ptr, 0) != cudaSuccess || dp != ptr) {
        cudaGetLastError();
        cudaHostUnregister(ptr);
        return fail(AES_E_CUDA);
    }
    return AES_OK;
}
extern "C" int aes_host_unregister(void *ptr)
{
    if (!ptr) return fail(AES_E_INVAL);
    if (cudaHostUnregister(ptr) != cudaSuccess) {
        cudaGetLastError();
        return fail(AES_E_INVAL);
    }
    return AES_OK;
}

/* ============================================================================================ */
/* launch backend: the paper's mechanism (own stream + event)                      */
/* ============================================================================================ */
namespace {
/* Everything one launch reads travels in ONE host->device copy: a blob of
 *   counters (256 B) | n descriptors | one expanded key per distinct context | the tickets
 * staged in pinned memory and mirrored at the same offsets in device memory.                     */
struct LaunchCtx {
    std::mutex mu;
    int device = -1;
    size_t cap_req = 0, cap_tickets = 0; /* capacities (power of two) */
    uint8_t *blob = nullptr;             /* device */
    uint8_t *stage = nullptr;            /* pinned host mirror */
    size_t blob_bytes = 0;
    uint64_t *dev_done_seq = nullptr;
    uint32_t *dq_done = nullptr, *dT0 = nullptr;
    cudaEvent_t stage_free = nullptr;
    bool stage_busy = false;
    /* The device blob (counters, descriptors, keys, tickets) is shared by all calls: a call on another stream
     * must not overwrite it while the previous call's kernel still reads it.  Every call makes its stream wait
     * for the previous call's kernel (one event), so calls from any streams are serialised on the device
     * in call order -- the payload of one launch fills the GPU anyway.                                    */
    cudaEvent_t kernel_done = nullptr;
    bool kernel_pending = false;
};
LaunchCtx g_lc;

size_t pow2_at_least(size_t x)
{
    size_t p = 64;
    while (p < x) p <<= 1;
    return p;
}
} /* namespace */

extern "C" int aes_ctr_launch_batch(aes_ctx_t *const *ctxs, const uint8_t *nonces, const void *const *srcs,
                                    void *const *dsts, const size_t *lens, size_t n, int device, void *cuda_stream,
                                    uint32_t chunk_rows)
{
    return aes_mode_launch_batch(nullptr, ctxs, nonces, srcs, dsts, lens, n, device, cuda_stream, chunk_rows);
}

extern "C" int aes_mode_launch_batch(const int32_t *modes, aes_ctx_t *const *ctxs, const uint8_t *nonces,
                                     const void *const *srcs, void *const *dsts, const size_t *lens, size_t n, int device,
                                     void *cuda_stream, uint32_t chunk_rows)
{
    if (n == 0) return AES_OK;
    if (!ctxs || !nonces || !srcs || !dsts || !lens) return fail(AES_E_INVAL);
    if (chunk_rows == 0) chunk_rows = 4;
    if (chunk_rows > 64 || !is_pow2(chunk_rows)) return fail(AES_E_INVAL);
    bool need_dec = false;
    for (size_t i = 0; modes && i < n; ++i) {
        if (modes[i] < AES_MODE_CTR || modes[i] > AES_MODE_CBC_DEC) return fail(AES_E_INVAL);
        if (modes[i] != AES_MODE_CTR && (lens[i] & 15u)) return fail(AES_E_INVAL);
        if (modes[i] == AES_MODE_CBC_DEC && lens[i] && srcs[i] == dsts[i]) return fail(AES_E_OVERLAP);
        need_dec = need_dec || modes[i] == AES_MODE_ECB_DEC || modes[i] == AES_MODE_CBC_DEC;
    }
    if (device >= 0 && device < AESOFF_MAX_DEVICES && g_engs[device].running.load()) return fail(AES_E_BUSY);
    for (size_t i = 0; i < n; ++i) {
        if (!ctxs[i]) return fail(AES_E_INVAL);
        const int rc = check_buffers(srcs[i], dsts[i], lens[i]);
        if (rc != AES_OK) return fail(rc);
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return fail(AES_E_CUDA);
    AesoffDeviceScope on_device(device); /* the caller's current device is restored on every return below */
    if (!on_device.ok) return fail(AES_E_CUDA);
    int sms = 0, major = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device);
    if (major != 10) return fail(AES_E_CUDA);
    cudaStream_t stream = (cudaStream_t)cuda_stream;

    LaunchCtx &L = g_lc;
    std::lock_guard<std::mutex> lk(L.mu);

    /* geometry first: how many tickets in all */
    const size_t R = pow2_at_least(n);
    std::vector<uint64_t> rows(n);
    std::vector<uint32_t> crows(n), nch(n);
    uint64_t total = 0;
    for (size_t i = 0; i < n; ++i) {
        /* rows are aligned on counter byte 15 being 0 in CTR mode, on the start of the payload otherwise */
        request_geometry(lens[i], (modes && modes[i]) ? 0 : nonces[16 * i + 15], chunk_rows, 1u << 24, &rows[i], &crows[i], &nch[i]);
        total += nch[i];
    }
    if (total >= (1ull << 30)) return fail(AES_E_INVAL);
    const size_t TM = pow2_at_least((size_t)total);

    /* (re)allocate the device blob and its pinned mirror */
    if (L.device != device || L.cap_req < R || L.cap_tickets < TM) {
        if (L.stage_busy) cudaEventSynchronize(L.stage_free);
        L.stage_busy = false;
        if (L.kernel_pending) cudaEventSynchronize(L.kernel_done);
        L.kernel_pending = false;
        if (L.blob) cudaFree(L.blob);
        if (L.dev_done_seq) cudaFree(L.dev_done_seq);
        if (L.dq_done) cudaFree(L.dq_done);
        if (L.dT0) cudaFree(L.dT0);
        if (L.stage) {
            explicit_bzero(L.stage, L.blob_bytes); /* key hygiene: expanded keys were staged here */
            cudaFreeHost(L.stage);
        }
        if (!L.stage_free) cudaEventCreateWithFlags(&L.stage_free, cudaEventDisableTiming);
        if (!L.kernel_done) cudaEventCreateWithFlags(&L.kernel_done, cudaEventDisableTiming);
        L.blob = nullptr;
        L.cap_req = R > L.cap_req ? R : L.cap_req;
        L.cap_tickets = TM > L.cap_tickets ? TM : L.cap_tickets;
        L.blob_bytes = AESOFF_CNT_WORDS * 8 + L.cap_req * (sizeof(aesoff_dq_entry_t) + sizeof(aesoff_key_t)) +
                       L.cap_tickets * sizeof(aesoff_ticket_t);
        bool ok = true;
        ok = ok && cudaMalloc((void **)&L.blob, L.blob_bytes) == cudaSuccess;
        ok = ok && cudaMalloc((void **)&L.dev_done_seq, L.cap_req * 8) == cudaSuccess;
        ok = ok && cudaMalloc((void **)&L.dq_done, L.cap_req * 4) == cudaSuccess;
        ok = ok && cudaMalloc((void **)&L.dT0, 512 * 4) == cudaSuccess;
        ok = ok && cudaHostAlloc((void **)&L.stage, L.blob_bytes, cudaHostAllocDefault) == cudaSuccess;
        ok = ok && cudaMemcpy(L.dT0, aesoff_T0_table(), 512 * 4, cudaMemcpyHostToDevice) == cudaSuccess;
        ok = ok && cudaMemset(L.dq_done, 0, L.cap_req * 4) == cudaSuccess;
        ok = ok && cudaMemset(L.dev_done_seq, 0, L.cap_req * 8) == cudaSuccess;
        if (!ok) {
            cudaGetLastError();
            L.device = -1;
            L.cap_req = L.cap_tickets = 0;
            return fail(AES_E_NOMEM);
        }
        L.device = device;
    }
    /* the previous call's copy must have left the staging buffer */
    if (L.stage_busy) {
        cudaEventSynchronize(L.stage_free);
        L.stage_busy = false;
    }
    /* blob layout for this call (every part a multiple of 16 bytes) */
    const size_t off_dq = AESOFF_CNT_WORDS * 8;
    const size_t off_key = off_dq + n * sizeof(aesoff_dq_entry_t);
    uint64_t *hc = reinterpret_cast<uint64_t *>(L.stage);
    std::vector<aesoff_dev_desc_t> hd(n); /* packed into tagged dq entries below */
    aesoff_dq_entry_t *hq = reinterpret_cast<aesoff_dq_entry_t *>(L.stage + off_dq);
    aesoff_key_t *hk = reinterpret_cast<aesoff_key_t *>(L.stage + off_key);
    size_t nkeys = 0;
    for (size_t i = 0; i < n; ++i) {
        /* one key entry per run of requests with the same context (host-expanded, aesoff_keys.cpp) */
        if (i == 0 || ctxs[i] != ctxs[i - 1]) {
            memset(&hk[nkeys], 0, sizeof(aesoff_key_t));
            host_round_keys(ctxs[i]);
            memcpy(hk[nkeys].rk, ctxs[i]->rk, sizeof(hk[nkeys].rk));
            ++nkeys;
        }
        aesoff_dev_desc_t &d = hd[i];
        memset(&d, 0, sizeof(d));
        memcpy(d.icb, nonces + 16 * i, 16);
        d.src = (uint64_t)(uintptr_t)srcs[i];
        d.dst = (uint64_t)(uintptr_t)dsts[i];
        d.len = (uint64_t)lens[i];
        d.nr = (uint32_t)ctxs[i]->nr;
        d.flags = modes ? (uint32_t)modes[i] : AESOFF_MODE_CTR;
        d.nchunks = nch[i];
        d.chunk_rows = crows[i];
        d.seq = i + 1;
        d.rows = rows[i];
        d.keyloc = (uint32_t)(nkeys - 1);
    }
    const size_t off_tk = off_key + nkeys * sizeof(aesoff_key_t);
    aesoff_ticket_t *ht = reinterpret_cast<aesoff_ticket_t *>(L.stage + off_tk);
    /* The end of a launch is the one place where big units cost: a warp's last row takes 10 us while
     * the rest of the GPU idles.  The chunks holding the last wave of rows (one row per worker warp)
     * are therefore cut into 1/8 rows and the four waves before them into half rows.               */
    uint64_t all_rows = 0;
    for (size_t i = 0; i < n; ++i) all_rows += rows[i];
    const uint64_t wave = (uint64_t)sms * AESOFF_WORKER_WARPS;
    uint64_t t = 0, rows_before = 0;
    for (size_t i = 0; i < n; ++i) {
        hd[i].first_ticket = t;
        for (uint32_t c = 0; c < nch[i]; ++c) {
            aesoff_ticket_t &tk = ht[t + c];
            const uint64_t left = all_rows - (rows_before + (uint64_t)c * crows[i]); /* rows from this chunk on */
            const uint32_t mode = left <= wave ? AESOFF_FLAG_FINE : left <= 5 * wave ? AESOFF_FLAG_HALF : 0u;
            tk.seq32 = (uint32_t)(i + 1);
            tk.chunk = c | (mode << AESOFF_TICKET_MODE_SHIFT);
            tk.keyloc = hd[i].keyloc;
            tk.tag = (uint32_t)(t + c) + 1u;
        }
        t += nch[i];
        rows_before += rows[i];
    }
    for (size_t i = 0; i < n; ++i) { /* the 24 descriptor words as 8 pieces of {3 words, tag = seq} */
        const uint32_t *w = reinterpret_cast<const uint32_t *>(&hd[i]);
        for (int q = 0; q < 8; ++q) {
            hq[i].w[4 * q + 0] = w[3 * q + 0];
            hq[i].w[4 * q + 1] = w[3 * q + 1];
            hq[i].w[4 * q + 2] = w[3 * q + 2];
            hq[i].w[4 * q + 3] = (uint32_t)(i + 1);
        }
    }
    memset(hc, 0, AESOFF_CNT_WORDS * 8);
    hc[AESOFF_CNT_PUBLISHED] = total;
#ifdef AESOFF_DEBUG
    hc[20] = hc[23] = hc[26] = ~0ull; /* the atomicMin stamps */
#endif
    const size_t used = off_tk + (size_t)total * sizeof(aesoff_ticket_t);

    bool ok = true;
    if (L.kernel_pending) ok = cudaStreamWaitEvent(stream, L.kernel_done, 0) == cudaSuccess;
    ok = ok && cudaMemcpyAsync(L.blob, L.stage, used, cudaMemcpyHostToDevice, stream) == cudaSuccess;
    ok = ok && cudaEventRecord(L.stage_free, stream) == cudaSuccess;
    L.stage_busy = true;
    if (!ok) {
        cudaGetLastError();
        return fail(AES_E_CUDA);
    }
    if (total == 0) return AES_OK;

    aesoff_params_t p;
    memset(&p, 0, sizeof(p));
    p.counters = reinterpret_cast<uint64_t *>(L.blob);
    p.dq = reinterpret_cast<aesoff_dq_entry_t *>(L.blob + off_dq);
    p.ktab = reinterpret_cast<aesoff_key_t *>(L.blob + off_key);
    p.tmap = reinterpret_cast<aesoff_ticket_t *>(L.blob + off_tk);
    p.dq_done = L.dq_done;
    p.dev_done_seq = L.dev_done_seq;
    p.T0 = L.dT0;
    p.drain_total = total;
    p.R = (uint32_t)R;
    p.TM = (uint32_t)L.cap_tickets;
    p.chunk_rows = chunk_rows;
    p.mode = AESOFF_MODE_DRAIN;
    p.need_dec = need_dec ? 1u : 0u;
    p.first_seq = 1;
    uint64_t total_rows = 0;
    for (size_t i = 0; i < n; ++i) total_rows += rows[i];
    uint64_t ctas = (total_rows + AESOFF_ROWS_PER_CTA - 1) / AESOFF_ROWS_PER_CTA;
    if (ctas > (uint64_t)sms) ctas = (uint64_t)sms;
    if (ctas == 0) ctas = 1;
    if (aesoff_launch_engine(&p, (int)ctas, stream) != 0) return fail(AES_E_CUDA);
    L.kernel_pending = cudaEventRecord(L.kernel_done, stream) == cudaSuccess;
    g_kernel_launches.fetch_add(1);
    return AES_OK;
}

#ifdef AESOFF_DEBUG
/* time stamps of the last launch (globaltimer ns): see DBG_MIN / DBG_MAX in aesoff_kernels.cu */
extern "C" __attribute__((visibility("default"))) int aesoff_debug_stamps(uint64_t out[8])
{
    LaunchCtx &L = g_lc;
    cudaDeviceSynchronize();
    return cudaMemcpy(out, L.blob + 20 * 8, 64, cudaMemcpyDeviceToHost) == cudaSuccess ? 0 : -1;
}
#endif

/* ============================================================================================ */
/* closed-loop executor (PAPER.md:127-135 worker loop; "50 concurrent clients")      */
/* ============================================================================================ */
namespace {
/* Per-request time stamps of the executors: two clock_gettime calls per request are half of what a 4 KiB
 * request costs the submitting thread, so on x86 the loops read the time stamp counter and convert with a
 * factor measured once against CLOCK_MONOTONIC_RAW.                                                     */
struct TickClock {
    double ns_per_tick = 1.0;
    TickClock()
    {
#if defined(__x86_64__)
        const uint64_t t0 = now_ns(), c0 = __rdtsc();
        while (now_ns() - t0 < 2000000ull) CPU_RELAX();
        const uint64_t t1 = now_ns(), c1 = __rdtsc();
        ns_per_tick = (double)(t1 - t0) / (double)(c1 - c0);
#endif
    }
};
inline uint64_t ticks()
{
#if defined(__x86_64__)
    return __rdtsc();
#else
    return now_ns();
#endif
}
inline double tick_ns()
{
    static const TickClock clk;
    return clk.ns_per_tick;
}
} /* namespace */

extern "C" int aes_loop_run(const aes_loop_spec_t *spec, aes_loop_result_t *res, double *lat_ns)
{
    if (!spec || !res || !spec->nonces || !spec->srcs || !spec->dsts || !spec->lens) return fail(AES_E_INVAL);
    if (!spec->keys && !spec->ctx) return fail(AES_E_INVAL);
    if (spec->keys && !spec->keybits) return fail(AES_E_INVAL);
    if (spec->n == 0 || spec->window == 0 || spec->mode > AES_MODE_CBC_DEC) return fail(AES_E_INVAL);
    const uint32_t running = g_running_mask.load(std::memory_order_acquire);
    if (!running) return fail(AES_E_STOPPED);
    uint32_t ring_total = 0; /* what can be in flight over all engines */
    for (int d = 0; d < AESOFF_MAX_DEVICES; ++d)
        if ((running >> d) & 1u) ring_total += g_engs[d].R;
    const uint64_t repeat = spec->repeat ? spec->repeat : 1;
    const uint64_t total = (uint64_t)spec->n * repeat;
    const uint32_t window = spec->window > ring_total ? ring_total : spec->window;
    const double nspt = tick_ns();

    /* In flight, in submission order.  Completions come roughly in that order, so a sweep polls from the oldest
     * and gives up after 32 requests that are still pending (every eighth sweep looks at all of them): a window
     * of 256 costs a few polls per completion, not 256.  A request that completed out of order stays in the
     * queue as a tombstone until the ones before it are gone.                                              */
    struct Fly {
        aes_handle_t h;
        uint64_t t_submit;
        uint64_t index;
    };
    size_t cap = 64;
    while (cap < 4 * (size_t)window) cap <<= 1;
    std::vector<Fly> q(cap);
    uint64_t head = 0, tail = 0, sweep = 0;
    uint32_t n_fly = 0;
    uint64_t next = 0, done = 0, bytes = 0;
    memset(res, 0, sizeof(*res));

    const uint64_t t_begin = now_ns();
    while (done < total) {
        /* submit until the window is full */
        while (n_fly < window && next < total && tail - head < cap) {
            const size_t i = (size_t)(next % spec->n);
            aes_ctx_t *ctx = spec->ctx;
            if (spec->keys) {
                ctx = aes_ctx_create(spec->keys + 32 * i, spec->keybits[i]);
                if (!ctx) return t_last_error;
            }
            const uint64_t ts = lat_ns ? ticks() : 0;
            const aes_handle_t h = submit_mode(ctx, spec->mode, spec->nonces + 16 * i, spec->srcs[i], spec->dsts[i], spec->lens[i]);
            if (spec->keys) aes_ctx_destroy(ctx);
            if (h == 0) {
                if (t_last_error == AES_E_AGAIN) {
                    ++res->ring_full_spins;
                    break;
                }
                return t_last_error;
            }
            q[tail++ & (cap - 1)] = Fly{h, ts, next};
            if (++n_fly > res->max_in_flight) res->max_in_flight = n_fly;
            ++next;
        }
        /* poll from the oldest */
        const bool all = (++sweep & 7u) == 0;
        uint32_t pending = 0;
        for (uint64_t k = head; k < tail; ++k) {
            Fly &f = q[k & (cap - 1)];
            if (f.h == 0) continue; /* tombstone */
            const int r = aes_poll(f.h);
            if (r == 1) {
                if (lat_ns) lat_ns[f.index] = (double)(ticks() - f.t_submit) * nspt;
                bytes += spec->lens[f.index % spec->n];
                ++done;
                --n_fly;
                f.h = 0;
            } else if (r < 0) {
                return r;
            } else if (++pending >= 32u && !all) {
                break;
            }
        }
        while (head < tail && q[head & (cap - 1)].h == 0) ++head;
    }
    res->elapsed_ns = now_ns() - t_begin;
    res->bytes = bytes;
    res->requests = done;
    return AES_OK;
}

/* ============================================================================================ */
/* calibration microkernels (aesoff_calib.cu)                                                     */
/* ============================================================================================ */
extern "C" int aes_calibrate(int device, aes_calib_t *out)
{
    if (!out) return fail(AES_E_INVAL);
    if (device >= 0 && device < AESOFF_MAX_DEVICES && g_engs[device].running.load()) return fail(AES_E_BUSY);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return fail(AES_E_CUDA);
    double v[8];
    if (aesoff_run_calibration(device, v) != 0) return fail(AES_E_CUDA);
    out->lookups_per_clk_per_sm = v[0] * 32.0; /* the kernel counts warp-wide LDS instructions */
    out->alu_instr_per_clk_per_sm = v[1];
    out->copy_gbs = v[2];
    out->sm_mhz = v[3];
    out->sm_count = (int32_t)v[4];
    out->reserved = 0;
    out->round_lookups_per_clk_per_sm = v[5] * 32.0;
    out->bitslice_sboxes_per_clk_per_sm = v[6];
    out->bitslice_mismatches = (int32_t)v[7];
    out->reserved2 = 0;
    return AES_OK;
}

/* ============================================================================================ */
/* open-loop executor (Fig. 12: Poisson arrivals, blocking vs overlapping)          */
/* ============================================================================================ */
extern "C" int aes_openloop_run(const aes_loop_spec_t *spec, const uint64_t *arrival_ns, int blocking,
                                aes_loop_result_t *res, double *lat_ns)
{
    if (!spec || !res || !arrival_ns || !spec->ctx || !spec->nonces || !spec->srcs || !spec->dsts || !spec->lens)
        return fail(AES_E_INVAL);
    if (spec->n == 0) return fail(AES_E_INVAL);
    if (!g_running_mask.load(std::memory_order_acquire)) return fail(AES_E_STOPPED);
    const size_t n = spec->n;
    struct Fly {
        aes_handle_t h;
        size_t index;
    };
    std::vector<Fly> fly;
    fly.reserve(4096);
    memset(res, 0, sizeof(*res));
    size_t next = 0, done = 0;
    uint64_t bytes = 0;
    const uint64_t t0 = now_ns();
    while (done < n) {
        uint64_t now = now_ns() - t0;
        /* every request whose arrival time has passed is submitted (the ring bounds what is in flight) */
        while (next < n && arrival_ns[next] <= now) {
            const aes_handle_t h = aes_ctr_submit(spec->ctx, spec->nonces + 16 * next, spec->srcs[next], spec->dsts[next],
                                                  spec->lens[next]);
            if (h == 0) {
                if (t_last_error == AES_E_AGAIN) {
                    ++res->ring_full_spins;
                    break;
                }
                return t_last_error;
            }
            if (blocking) {
                /* the server that waits for its offload: nothing else is served meanwhile */
                const int rc = aes_wait(h, UINT64_MAX);
                if (rc != AES_OK) return rc;
                now = now_ns() - t0;
                if (lat_ns) lat_ns[next] = (double)(now - arrival_ns[next]);
                bytes += spec->lens[next];
                ++done;
            } else {
                fly.push_back(Fly{h, next});
                if (fly.size() > res->max_in_flight) res->max_in_flight = fly.size();
            }
            ++next;
        }
        size_t k = 0;
        while (k < fly.size()) {
            const int r = aes_poll(fly[k].h);
            if (r == 1) {
                if (lat_ns) lat_ns[fly[k].index] = (double)(now_ns() - t0 - arrival_ns[fly[k].index]);
                bytes += spec->lens[fly[k].index];
                ++done;
                fly[k] = fly.back();
                fly.pop_back();
            } else if (r < 0) {
                return r;
            } else {
                ++k;
            }
        }
    }
    res->elapsed_ns = now_ns() - t0;
    res->bytes = bytes;
    res->requests = done;
    return AES_OK;
}

/* ============================================================================================ */
/* closed loop from several executor threads ("worker pool")           */
/* ============================================================================================ */
extern "C" int aes_loop_run_mt(const aes_loop_spec_t *spec, uint32_t nthreads, aes_loop_result_t *res, double *lat_ns)
{
    if (!spec || !res || nthreads == 0 || nthreads > 64) return fail(AES_E_INVAL);
    if (spec->n < nthreads) return fail(AES_E_INVAL);
    std::vector<aes_loop_spec_t> specs(nthreads, *spec);
    std::vector<aes_loop_result_t> results(nthreads);
    std::vector<int> rcs(nthreads, AES_OK);
    std::vector<std::thread> threads;
    const size_t per = spec->n / nthreads;
    const uint32_t window = spec->window / nthreads ? spec->window / nthreads : 1u;
    const uint64_t t0 = now_ns();
    for (uint32_t t = 0; t < nthreads; ++t) {
        aes_loop_spec_t &s = specs[t];
        const size_t first = per * t, count = (t + 1 == nthreads) ? spec->n - first : per;
        s.n = count;
        s.window = window;
        s.nonces = spec->nonces + 16 * first;
        s.srcs = spec->srcs + first;
        s.dsts = spec->dsts + first;
        s.lens = spec->lens + first;
        if (spec->keys) {
            s.keys = spec->keys + 32 * first;
            s.keybits = spec->keybits + first;
        }
        double *lat = lat_ns ? lat_ns + first * (spec->repeat ? spec->repeat : 1) : nullptr;
        threads.emplace_back([&, t, lat]() {
            rcs[t] = aes_loop_run(&specs[t], &results[t], lat);
            if (rcs[t] != AES_OK) rcs[t] = t_last_error ? t_last_error : rcs[t];
        });
    }
    for (auto &th : threads) th.join();
    memset(res, 0, sizeof(*res));
    res->elapsed_ns = now_ns() - t0;
    for (uint32_t t = 0; t < nthreads; ++t) {
        if (rcs[t] != AES_OK) return fail(rcs[t]);
        res->bytes += results[t].bytes;
        res->requests += results[t].requests;
        res->ring_full_spins += results[t].ring_full_spins;
        res->max_in_flight += results[t].max_in_flight;
    }
    return AES_OK;
}

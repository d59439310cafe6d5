/*
 * aesoff_router.cpp -- which engine a request goes to when several GPUs of a node each run one
 * (SURVEY.md section 8(e) and (f4)).  Requests are independent ("each offload belongs to one request",
 * PAPER.md:25, 105-107) and so are the blocks inside one: the path shards with NO exchange step, so the
 * router is a table look-up, not a collective:
 *
 *   - device memory decides: a request runs on the GPU that owns its device buffer(s); moving a payload over
 *     NVLink to encrypt it elsewhere would cost about what the cipher does;
 *   - src on one GPU and dst on another is refused (AESOFF_ROUTE_MIXED): an engine's kernel dereferences both,
 *     and this library never enables peer access, so whichever engine took it would fault and lose all it holds;
 *   - a request whose src and dst are both host memory (the paper's j.buf) may run anywhere:
 *     the running engines take such requests in turn;
 *   - with ONE engine running on a node with ONE GPU everything goes there and no address is looked at.
 *
 * Owners are resolved by the caller's function (cudaPointerGetAttributes in the runtime, a table in the CPU
 * tests) and remembered per 2 MiB page in a small per-thread cache: allocations of different devices never
 * share a 2 MiB page of the unified address space.  A page that is freed and handed to another device needs
 * aes_route_flush() (include/aesoff.h).  No cipher arithmetic here; no CUDA call either.
 */
#include <stdint.h>

#include <atomic>

#include "aesoff_internal.h"

int aesoff_route_decide(int src_owner, int dst_owner, uint32_t running_mask, uint32_t *round_robin)
{
    if (running_mask == 0) return AESOFF_ROUTE_NONE;
    if (src_owner >= 0 && dst_owner >= 0 && src_owner != dst_owner) return AESOFF_ROUTE_MIXED;
    if (dst_owner >= 0) return ((running_mask >> dst_owner) & 1u) ? dst_owner : -1; /* its owner has no engine: refuse */
    if (src_owner >= 0) return ((running_mask >> src_owner) & 1u) ? src_owner : -1;
    /* host memory on both sides: the running engines in turn */
    const uint32_t n = (uint32_t)__builtin_popcount(running_mask);
    uint32_t k = (*round_robin)++ % n;
    for (int d = 0; d < AESOFF_MAX_DEVICES; ++d)
        if ((running_mask >> d) & 1u) {
            if (k == 0) return d;
            --k;
        }
    return -1;
}

namespace {
std::atomic<uint32_t> g_generation{1};
struct PageCache {
    static constexpr int N = 64;
    uint64_t page[N];
    int owner[N];
    uint32_t generation = 0;
};
thread_local PageCache t_cache;
} /* namespace */

void aesoff_route_flush_cache(void) { g_generation.fetch_add(1, std::memory_order_release); }

int aesoff_route_owner_cached(const void *ptr, aesoff_owner_fn resolve)
{
    PageCache &c = t_cache;
    const uint32_t gen = g_generation.load(std::memory_order_acquire);
    if (c.generation != gen) {
        for (int i = 0; i < PageCache::N; ++i) c.page[i] = ~0ull;
        c.generation = gen;
    }
    const uint64_t page = (uint64_t)(uintptr_t)ptr >> 21;
    const int slot = (int)((page ^ (page >> 6) ^ (page >> 12)) & (PageCache::N - 1));
    if (c.page[slot] == page) return c.owner[slot];
    const int o = resolve(ptr);
    c.page[slot] = page;
    c.owner[slot] = o;
    return o;
}

/* ---- hooks for the CPU tests (tests/test_router_cpu.py): the same two functions over a synthetic address map ---- */
namespace {
thread_local uint64_t t_resolver_calls = 0;
/* addresses with bit 40 set are "device memory" of device (addr >> 30) & 7, everything else is host memory */
int synthetic_owner(const void *ptr)
{
    ++t_resolver_calls;
    const uint64_t a = (uint64_t)(uintptr_t)ptr;
    return (a >> 40) & 1u ? (int)((a >> 30) & 7u) : AESOFF_OWNER_HOST;
}
} /* namespace */

extern "C" __attribute__((visibility("default"))) int aesoff_test_route_decide(int src_owner, int dst_owner, uint32_t running_mask,
                                                                               uint32_t *round_robin)
{
    return aesoff_route_decide(src_owner, dst_owner, running_mask, round_robin);
}

/* routes n (src, dst) pairs over the synthetic map; returns how often the resolver had to be asked */
extern "C" __attribute__((visibility("default"))) uint64_t aesoff_test_route_many(const uint64_t *srcs, const uint64_t *dsts, size_t n,
                                                                                  uint32_t running_mask, int32_t *out, int flush_first)
{
    if (flush_first) aesoff_route_flush_cache();
    t_resolver_calls = 0;
    uint32_t rr = 0;
    for (size_t i = 0; i < n; ++i) {
        const int dO = aesoff_route_owner_cached((const void *)(uintptr_t)dsts[i], synthetic_owner);
        const int so = aesoff_route_owner_cached((const void *)(uintptr_t)srcs[i], synthetic_owner);
        out[i] = aesoff_route_decide(so, dO, running_mask, &rr);
    }
    return t_resolver_calls;
}

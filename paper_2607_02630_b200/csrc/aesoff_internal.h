/* aesoff_internal.h -- declarations shared by the host translation units (internal). */
#ifndef AESOFF_INTERNAL_H
#define AESOFF_INTERNAL_H

#include <stdint.h>

#include "aesoff_shared.h"

/* How a context's key reaches the device (aesoff_runtime.cpp, aes_ctr_submit):
 *   first submit        the raw key rides in the descriptor, the dispatcher that takes the request
 *                       expands it (one-shot contexts, BASELINE.json configs[3], never own device state)
 *   second submit       as above, and that dispatcher also stores the expanded key at ktab[id]
 *   until that request has COMPLETED (mailbox)   raw key again, nothing stored: several dispatcher warps
 *                       take requests side by side, so "submitted earlier" does not mean "expanded earlier"
 *   afterwards          the descriptor only names ktab[id]
 * An id belongs to one generation of the key table (epoch): INSTALLED or INSTALLING under an older epoch starts over. */
#define AESOFF_CTX_FRESH      0u
#define AESOFF_CTX_SEEN       1u
#define AESOFF_CTX_INSTALLING 2u
#define AESOFF_CTX_INSTALLED  3u
#define AESOFF_CTX_CLAIMED    4u /* transient: one thread is writing id / epoch / install_seq on its way to INSTALLING */

#define AESOFF_MAX_DEVICES 8 /* engines per process: one per GPU of a node */

/* where a context's key is on ONE engine (each GPU has its own key table) */
struct aes_ctx_dev {
    uint32_t state;       /* AESOFF_CTX_*, accessed atomically */
    uint32_t id;          /* ktab index once state >= INSTALLING */
    uint64_t epoch;       /* ktab generation the id belongs to */
    uint64_t install_seq; /* sequence number of the request that installs the key (0 = not claimed yet) */
};

struct aes_ctx {
    uint32_t rk[60]; /* round keys as little-endian-loaded words, zero padded (host expansion) */
    int32_t nr;      /* 10, 12 or 14 */
    int32_t keybits;
    uint32_t key[8]; /* the cipher key as little-endian-loaded words, zero padded */
    uint32_t rk_ready; /* rk[] has been filled (lazily: the engine path expands keys on the device) */
    uint32_t pad_;
    aes_ctx_dev dev[AESOFF_MAX_DEVICES];
};

/* Which engine a request goes to (aesoff_router.cpp; "requests routed to the GPU that owns
 * their src/dst").  owner: device index of the memory, AESOFF_OWNER_HOST for host memory.                        */
#define AESOFF_OWNER_HOST (-2)
#define AESOFF_ROUTE_NONE  (-1) /* aesoff_route_decide: nothing runs, or the owner of the memory runs no engine */
#define AESOFF_ROUTE_MIXED (-2) /* src and dst belong to two different GPUs */
int aesoff_route_decide(int src_owner, int dst_owner, uint32_t running_mask, uint32_t *round_robin);
typedef int (*aesoff_owner_fn)(const void *ptr); /* resolves the owner of an address (cudaPointerGetAttributes) */
int aesoff_route_owner_cached(const void *ptr, aesoff_owner_fn resolve);
void aesoff_route_flush_cache(void);

/* Makes `device` current for a scope and puts the caller's device back at its end: a process that runs torch (or an
 * engine) on another GPU must not find its later allocations moved because it called into this library.        */
#ifdef __CUDA_RUNTIME_H__
struct AesoffDeviceScope {
    int prev = -1, target = -1;
    bool ok = false;
    explicit AesoffDeviceScope(int device) : target(device)
    {
        ok = cudaGetDevice(&prev) == cudaSuccess && (prev == device || cudaSetDevice(device) == cudaSuccess);
    }
    ~AesoffDeviceScope()
    {
        if (ok && prev != target) cudaSetDevice(prev);
    }
    AesoffDeviceScope(const AesoffDeviceScope &) = delete;
    AesoffDeviceScope &operator=(const AesoffDeviceScope &) = delete;
};
#endif

const uint32_t *aesoff_T0_table();
int aesoff_key_expand(const uint8_t *key, int keybits, uint32_t rk[60]);

extern "C" int aesoff_launch_engine(const aesoff_params_t *params, int n_ctas, void *stream);
extern "C" int aesoff_run_calibration(int device, double out[8]);

#endif

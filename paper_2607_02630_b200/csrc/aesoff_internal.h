/* aesoff_internal.h -- declarations shared by the host translation units (internal). */
#ifndef AESOFF_INTERNAL_H
#define AESOFF_INTERNAL_H

#include <stdint.h>

#include "aesoff_shared.h"

struct aes_ctx {
    uint32_t rk[60]; /* round keys as little-endian-loaded words, zero padded */
    int32_t nr;      /* 10 or 14 */
    int32_t keybits;
};

const uint32_t *aesoff_T0_table();
int aesoff_key_expand(const uint8_t *key, int keybits, uint32_t rk[60]);

extern "C" int aesoff_launch_engine(const aesoff_params_t *params, int n_ctas, void *stream);

#endif

/* readgen_host.c — host twin of the synthetic read generator (see readgen_core.h). Input generation only. */
#include "readgen_core.h"

/* Writes reads [r0, r1) as ASCII, read r at out[(r-r0)*L .. +L). */
void rg_generate_host(const rg_params *p, const uint64_t *glen, const uint64_t *cdf,
                      uint64_t r0, uint64_t r1, char *out) {
    const uint32_t L = p->read_len;
    for (uint64_t r = r0; r < r1; ++r) {
        rg_read h = rg_read_header(p, glen, cdf, r);
        char *o = out + (r - r0) * (uint64_t)L;
        for (uint32_t j = 0; j < L; ++j) o[j] = rg_read_letter(p, &h, j);
    }
}

uint64_t rg_hash_host(uint64_t seed, uint64_t stream, uint64_t a, uint64_t b) { return rg_hash(seed, stream, a, b); }

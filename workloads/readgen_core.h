/* readgen_core.h — seeded, counter-based synthetic read generator (shared by the host twin
 * readgen_host.c and the device twin readgen_cuda.cu, so both produce identical bytes).
 *
 * This is INPUT GENERATION ONLY: it holds none of the SdBG method's arithmetic (no 2-bit packing,
 * no k-mer keys, no sorting). It writes ASCII reads over {A,C,G,T}; both the CPU oracle and the
 * CUDA library consume those bytes. Recipe: SURVEY.md §8(d) / DESIGN.md "Input recipe"; the
 * workloads stand in for the paper's E. coli and soil read sets.
 *
 *   mix(z)            : splitmix64 finaliser
 *   hash(seed,s,a,b)  : mix(mix(mix(seed ^ mix(s+1)) + a) + b)        (s = stream id)
 *   genome base(g,p)  : 2 bits of hash(seed, GENOME, g, p>>5) at bit offset 2*(p&31); genomes are
 *                       never materialised
 *   read r            : genome g = first index with cdf[g] >= hash(seed,READ,r,0)   (u64 CDF table)
 *                       start    = hash(seed,READ,r,1) mod (len[g]-L+1)
 *                       strand   = hash(seed,READ,r,2) & 1        (1 = reverse complement)
 *                       base j   = strand ? 3-base(g,start+L-1-j) : base(g,start+j)
 *                       error j  : e = mix(hash(seed,ERR,r,0) + j);  if (e>>32) < err_thr then
 *                                  base = (base + 1 + (e & 0xffffffff) mod 3) & 3
 *                       letter   = "ACGT"[base]
 */
#ifndef READGEN_CORE_H
#define READGEN_CORE_H
#include <stdint.h>

#ifdef __CUDACC__
#define RG_HD __host__ __device__ __forceinline__
#else
#define RG_HD static inline
#endif

#define RG_STREAM_GENOME 1ull
#define RG_STREAM_READ   2ull
#define RG_STREAM_ERR    3ull
#define RG_STREAM_TABLE  4ull

typedef struct {
    uint64_t seed;
    uint64_t n_genomes;
    uint32_t read_len;
    uint32_t err_thr;      /* floor(eps * 2^32) */
} rg_params;

RG_HD uint64_t rg_mix(uint64_t z) {
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    return z;
}

RG_HD uint64_t rg_hash(uint64_t seed, uint64_t stream, uint64_t a, uint64_t b) {
    uint64_t h = rg_mix(seed ^ rg_mix(stream + 1));
    h = rg_mix(h + a);
    h = rg_mix(h + b);
    return h;
}

RG_HD uint32_t rg_genome_base(uint64_t seed, uint64_t g, uint64_t pos) {
    uint64_t w = rg_hash(seed, RG_STREAM_GENOME, g, pos >> 5);
    return (uint32_t)(w >> (2 * (pos & 31))) & 3u;
}

/* first index g in [0,n) with cdf[g] >= x; cdf[n-1] == UINT64_MAX so one always exists */
RG_HD uint64_t rg_pick_genome(const uint64_t *cdf, uint64_t n, uint64_t x) {
    uint64_t lo = 0, hi = n - 1;
    while (lo < hi) {
        uint64_t mid = lo + ((hi - lo) >> 1);
        if (cdf[mid] >= x) hi = mid; else lo = mid + 1;
    }
    return lo;
}

typedef struct { uint64_t g, start, errkey; uint32_t strand; } rg_read;

RG_HD rg_read rg_read_header(const rg_params *p, const uint64_t *glen, const uint64_t *cdf, uint64_t r) {
    rg_read h;
    h.g = rg_pick_genome(cdf, p->n_genomes, rg_hash(p->seed, RG_STREAM_READ, r, 0));
    h.start = rg_hash(p->seed, RG_STREAM_READ, r, 1) % (glen[h.g] - p->read_len + 1);
    h.strand = (uint32_t)(rg_hash(p->seed, RG_STREAM_READ, r, 2) & 1);
    h.errkey = rg_hash(p->seed, RG_STREAM_ERR, r, 0);
    return h;
}

RG_HD char rg_read_letter(const rg_params *p, const rg_read *h, uint32_t j) {
    uint32_t b = h->strand ? 3u - rg_genome_base(p->seed, h->g, h->start + p->read_len - 1 - j)
                           : rg_genome_base(p->seed, h->g, h->start + j);
    uint64_t e = rg_mix(h->errkey + j);
    if ((uint32_t)(e >> 32) < p->err_thr) b = (b + 1u + (uint32_t)(e & 0xffffffffu) % 3u) & 3u;
    return (char)((0x54474341u >> (8 * b)) & 0xff);   /* bytes 'A','C','G','T' */
}
#endif

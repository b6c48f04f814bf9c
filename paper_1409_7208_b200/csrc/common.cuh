// common.cuh — shared device/host helpers of libsdbg (sm_100a). Product code: never includes anything of oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

typedef unsigned long long u64;
typedef unsigned int u32;

namespace sdbg {

constexpr int kNumSMs = 148;           // B200; launch sizing uses num_sms(), read from the device in sdbg_ctx_create
extern int g_num_sms;
inline int num_sms() { return g_num_sms; }
constexpr int kMaxPasses = 32;         // 4 words x 8 digits
constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;

// One LSD pass: digit = (key.word[word] >> shift) & ((1 << bits) - 1).
struct PassDesc { uint8_t word, shift, bits, pad; };
struct PassTable { int n; PassDesc p[kMaxPasses]; };

// ---- tile status words for decoupled look-back -------------------------------------------------------
// [63:62] status, [61:54] epoch (onesweep only), [53:0] value.
constexpr u64 kStInvalid = 0ull, kStLocal = 1ull, kStGlobal = 2ull;

__device__ __forceinline__ u64 ld_relaxed(const u64 *p) {
    u64 v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed(u64 *p, u64 v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// streaming (evict-first) accesses for data touched once per pass
__device__ __forceinline__ u64 ld_stream(const u64 *p) {
    u64 v;
    asm volatile("ld.global.cs.u64 %0, [%1];" : "=l"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ uint2 ld_nc_u32x2(const void *p) {
    uint2 v;
    asm volatile("ld.global.nc.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
    return v;
}

__device__ __forceinline__ u32 lane_id() { return threadIdx.x & 31u; }
__device__ __forceinline__ u32 lanemask_lt() {
    u32 m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// splitmix64 finaliser; checksum definition in include/sdbg.h (sdbg_stats).
__device__ __forceinline__ u64 mix64(u64 z) {
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    return z;
}
template <int W>
__device__ __forceinline__ u64 mix_key(const u64 (&k)[W]) {
    u64 h = 0;
#pragma unroll
    for (int j = 0; j < W; ++j) h = mix64(h ^ k[j]);
    return h;
}

// one-word stand-in of a key of W > 1 words (kernels.cuh ExtractArgs::pair_keys): the top `top_bits` bits (8 .. 32) of the
// first word, so that stand-ins sort like keys as far as the top radix passes look, and below them a fingerprint of the
// whole key: the HIGH bits of the form  sum over the 32-bit halves w_i of  w_i * c_i + brev(w_i) * d_i  (mod 2^64).
// A product carries a bit of its factor upwards only, so w_i * c_i alone hardly sees the top bits of w_i; the bit-reversed
// copy sees exactly those. The extractor makes two fingerprints per window, so they must be cheap (one multiply-add per
// term), and the keys it meets are full of near-twins — every two copies of an edge with sequencing errors differ in a
// few symbols, and at 10^9 records every pattern of two or three changed symbols occurs — so no such pattern may cancel.
// Measured on config 4 (1.36 G records): a splitmix64 finaliser per word never met two keys but doubled the time of the
// extractor; sum(w_i * c_i) alone met thousands (2 c_1 - 12 c_4 happened to lie below 2^24); sum((w ^ (w >> 32)) * C_w)
// met the keys that differ in bits 62 and 30 of a word (the fold cancels them). For the form and the constants below all
// patterns of one, two and three changed symbols were enumerated (it is linear over Z / 2^64, so a pattern has ONE
// difference whatever the keys are): none comes closer than 2^30 (tests/test_fingerprint.py redoes it). Never all ones
// (the empty mark of the tables). Equal keys give equal stand-ins; the converse is CHECKED by the table count
// (hashcount.cu), which sends the range the plain way when two keys meet.
template <int W>
__device__ __forceinline__ u64 pair_key(const u64 (&k)[W], u32 top_bits, bool weak) {
    constexpr u32 c[8] = {0xbc91727fu, 0xc1835ef9u, 0xe0a95433u, 0xf9a8cb5du, 0x84760c67u, 0x9273d27bu, 0xe95637e9u, 0xf96d5857u};
    constexpr u32 d[8] = {0x9fe6b955u, 0xa7ea17d1u, 0xef3c3825u, 0xb62f8fa3u, 0xa2f73693u, 0xe9f22899u, 0xa0e51d65u, 0xb460a327u};
    static_assert(W <= 4, "eight pairs of constants");
    u64 h = 0;
#pragma unroll
    for (int q = 0; q < W; ++q) {
        const u32 lo = (u32)k[q], hi = (u32)(k[q] >> 32);
        h += (u64)lo * c[2 * q] + (u64)hi * c[2 * q + 1] + (u64)__brev(lo) * d[2 * q] + (u64)__brev(hi) * d[2 * q + 1];
    }
    const u64 low = ~0ull >> top_bits;
    const u64 fp = weak ? k[0] & low : h >> top_bits;
    const u64 p = (k[0] & ~low) | fp;
    return p == ~0ull ? p - 1ull : p;
}

__device__ __forceinline__ u32 warp_incl_scan_add(u32 v) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        u32 t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane_id() >= (u32)o) v += t;
    }
    return v;
}
__device__ __forceinline__ u64 warp_reduce_add64(u64 v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Statistics counters are spread over kStatSlots slots of one 128-byte line each (tile & 31 picks the slot), so that
// the one-atomic-per-block updates do not serialise on one L2 address; the host adds the slots up.
constexpr int kStatSlots = 32, kStatSlotWords = 16;   // words: 0 n_distinct, 1 sum_solid_mult, 2 csum_distinct

// ---- device-side scalars living at the start of the workspace -----------------------------------------
struct DevState {
    u64 bad_base;          // min index of a non-ACGT byte, ~0 if none
    u64 n_windows;         // valid (k+1)-windows in the packed reads
    u64 extract_cursor;    // records written by the extractor in this range
    u64 out_cursor[2];     // solid edges appended so far (may exceed cap: needed count); range r reads slot r&1, writes slot (r+1)&1
    u64 csum_raw;
    u64 merge_heads;       // sdbg_build unsorted path: distinct keys
    u32 tickets[kMaxPasses + 4];  // per-pass tile tickets; [kMaxPasses] = count kernel ticket
};

}  // namespace sdbg

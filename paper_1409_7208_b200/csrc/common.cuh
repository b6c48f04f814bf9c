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

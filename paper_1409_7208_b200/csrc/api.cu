// api.cu — the C ABI of include/sdbg.h: context, workspace layout, block-wise pass planner (step a6) and the
// sequencing of the kernels of pack.cu / extract.cu / radix.cu / count.cu / emit.cu. No device allocation happens
// here: everything lives in the caller's workspace. There is no CPU fallback.
#include "../../include/sdbg.h"
#include "kernels.cuh"

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

using namespace sdbg;

int sdbg::g_num_sms = sdbg::kNumSMs;   // replaced by the device's own count in sdbg_ctx_create

namespace {

constexpr u64 kAlign = 256;
inline u64 align_up(u64 x, u64 a = kAlign) { return (x + a - 1) / a * a; }
inline u64 *U64(uint64_t *p) { return reinterpret_cast<u64 *>(p); }
inline const u64 *U64C(const uint64_t *p) { return reinterpret_cast<const u64 *>(p); }

// fixed region at the start of the workspace
constexpr u64 kOffState = 0;
constexpr u64 kOffStatSlots = 1024;                                         // u64[kStatSlots][kStatSlotWords]
constexpr u64 kStatBytes = (u64)kStatSlots * kStatSlotWords * 8;
constexpr u64 kOffDigitHist = kOffStatSlots + kStatBytes;                   // u64[kMaxPasses][256]
constexpr u64 kOffBucketHist = kOffDigitHist + (u64)kMaxPasses * kRadix * 8;  // u64[65536]
constexpr u64 kFixedBytes = (kOffBucketHist + (u64)SDBG_NUM_BUCKETS * 8 + 4095) / 4096 * 4096;
static_assert(sizeof(DevState) <= 1024, "DevState must fit its slot");

struct EventPair { int cls; cudaEvent_t a, b; };
struct Fetch { void *dst; u64 off, bytes; };
constexpr u64 kFetchBytes = 64 * 1024;   // pinned, device-mapped host buffer of a context for small read-backs

// Small results (counters, flags, statistics) reach the host through stores of a kernel into mapped pinned memory,
// not through a device-to-host cudaMemcpyAsync: an asynchronous copy queues on the copy engine behind whatever
// bulk copy another stream of the process has in flight (the results of the previous step on their way to the host:
// measured 3.3 ms of waiting per read-back with 187 MB in flight), a store does not.
__global__ void fetch_kernel(const u64 *__restrict__ src, u64 *__restrict__ dst, u32 nwords) {
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < nwords; i += gridDim.x * blockDim.x) dst[i] = src[i];
}

}  // namespace

struct sdbg_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    char *ws = nullptr;
    u64 ws_bytes = 0;
    std::string err;
    bool timing = false;
    bool force_wide = false;   // SDBG_OPT_FORCE_WIDE (sdbg_ctx_set_option, include/sdbg.h)
    bool no_unstable = false;  // SDBG_OPT_STABLE_FIRST_PASS: the first radix pass uses the stable kernel like the others
    bool weak_fp = false;      // SDBG_OPT_WEAK_FINGERPRINT (tests)
    bool no_fused = false;     // SDBG_OPT_NO_FUSED_EXTRACT: the keys are written in read order and the first top pass reads them back
    bool no_hash = false;      // SDBG_OPT_NO_TABLE_COUNT: every record through every radix pass, then the sweeps of count.cu
    std::vector<EventPair> pending;
    std::vector<cudaEvent_t> free_events;
    char *fetch_buf = nullptr;   // kFetchBytes of mapped pinned host memory
    u64 fetch_used = 0;
    std::vector<Fetch> fetches;
    sdbg_timing acc{};

    DevState *st() const { return reinterpret_cast<DevState *>(ws + kOffState); }
    u64 *stat_slots() const { return reinterpret_cast<u64 *>(ws + kOffStatSlots); }
    u64 *digit_hist() const { return reinterpret_cast<u64 *>(ws + kOffDigitHist); }
    u64 *bucket_hist() const { return reinterpret_cast<u64 *>(ws + kOffBucketHist); }
    char *dyn() const { return ws + kFixedBytes; }
    u64 dyn_bytes() const { return ws_bytes > kFixedBytes ? ws_bytes - kFixedBytes : 0; }

    int fail(int code, const std::string &msg) { err = msg; return code; }
    int cuda_fail(cudaError_t e, const char *what) {
        err = std::string(what) + ": " + cudaGetErrorString(e);
        return SDBG_E_CUDA;
    }
    // enqueue: `bytes` (rounded up to 8; dev_src 8-byte aligned) of device memory -> host_dst, delivered by fetch_sync()
    int fetch(void *host_dst, const void *dev_src, u64 bytes) {
        const u64 words = (bytes + 7) / 8;
        if (fetch_used + words * 8 > kFetchBytes) { int rc = fetch_sync(); if (rc) return rc; }
        if (words * 8 > kFetchBytes) return fail(SDBG_E_INVAL, "internal: read-back larger than the fetch buffer");
        fetch_kernel<<<(unsigned)((words + 255) / 256), 256, 0, stream>>>(reinterpret_cast<const u64 *>(dev_src),
                                                                           reinterpret_cast<u64 *>(fetch_buf + fetch_used), (u32)words);
        fetches.push_back(Fetch{host_dst, fetch_used, bytes});
        fetch_used += words * 8;
        return SDBG_OK;
    }
    // synchronises the stream and hands every enqueued read-back to its destination
    int fetch_sync() {
        cudaError_t e = cudaStreamSynchronize(stream);
        if (e != cudaSuccess) { fetches.clear(); fetch_used = 0; return cuda_fail(e, "cudaStreamSynchronize"); }
        for (auto &f : fetches) memcpy(f.dst, fetch_buf + f.off, f.bytes);
        fetches.clear(); fetch_used = 0;
        return SDBG_OK;
    }
    cudaEvent_t get_event() {
        if (!free_events.empty()) { cudaEvent_t e = free_events.back(); free_events.pop_back(); return e; }
        cudaEvent_t e = nullptr;
        cudaEventCreate(&e);
        return e;
    }
};

namespace {

// RAII bracket of one kernel class: counts launches/bytes always, records events when timing is on.
struct Timed {
    sdbg_ctx *c; int cls; EventPair ep{};
    Timed(sdbg_ctx *c_, int cls_, u64 launches, u64 bytes) : c(c_), cls(cls_) {
        c->acc.launches[cls] += launches;
        c->acc.bytes[cls] += bytes;
        if (c->timing) { ep.cls = cls; ep.a = c->get_event(); ep.b = c->get_event(); cudaEventRecord(ep.a, c->stream); }
    }
    ~Timed() {
        if (c->timing) { cudaEventRecord(ep.b, c->stream); c->pending.push_back(ep); }
    }
};

#define RC(call)                                                        \
    do {                                                                \
        int rc__ = (call);                                              \
        if (rc__ != SDBG_OK) return rc__;                               \
    } while (0)

#define CU(call)                                                        \
    do {                                                                \
        cudaError_t e__ = (call);                                       \
        if (e__ != cudaSuccess) return ctx->cuda_fail(e__, #call);      \
    } while (0)

// LSD passes over the significant bits only, least significant first. Every digit is one whole byte of a key
// word (the sorter extracts it with a single byte-permute): the lowest pass starts at the byte that holds the first
// significant bit, and the zero padding bits below it simply leave some of its 256 bins empty.
PassTable make_passes(u32 k) {
    PassTable pt{};
    const u32 W = (2 * (k + 1) + 63) / 64;
    const u32 pad = 64 * W - 2 * (k + 1);
    for (int w = (int)W - 1; w >= 0; --w)
        for (u32 lo = (w == (int)W - 1) ? pad / 8 * 8 : 0; lo < 64; lo += kRadixBits)
            pt.p[pt.n++] = PassDesc{(uint8_t)w, (uint8_t)lo, (uint8_t)kRadixBits, 0};
    return pt;
}

bool is_device_ptr(const void *p) {
    cudaPointerAttributes at{};
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

// bytes of dynamic workspace a sort+count of n records needs (keys only)
// records per look-back row of the sorter that handles W-word keys: the keys themselves (W = 1) or (word, index) pairs
// records per radix tile, for the size of the look-back words: keys of several words go through pair passes (a key word
// and an index) or, on the table-count path, through passes over whole records: the smaller tile of the two
u64 sort_tile_records(u32 W) { return W == 1 ? radix_tile_records(1, false) : std::min(radix_tile_records(1, true), radix_tile_records(W, false)); }
// room behind the buffers of a range for the scratch of the table-count path (api_count.inc hash_scratch_bytes:
// segment borders and counts, 16 bytes per 2,048 records, block sums, a copy of the statistics)
u64 table_slack(u64 n, u32) { return align_up(n / 64) + kStatBytes + 16384; }
u64 range_need(u64 n, u32 W) {
    const u64 K = 8ull * W;
    const u64 rt = sort_tile_records(W), ct = count_tile_records(W);
    const u64 pairs = W == 1 ? 0 : 2 * align_up(n * 8) + 2 * align_up(n * 4);   // (word, index) ping-pong buffers
    return 2 * align_up(n * K) + pairs + align_up(((n + rt - 1) / rt + 1) * kRadix * 8) + align_up(((n + ct - 1) / ct + 1) * 8) + table_slack(n, W);
}
// largest n with range_need(n) <= avail; one sort range is also capped by the layout of the radix passes' look-back
// words (radix_max_records: 2^34-1 records or 2^22 tiles); larger inputs are split into block-wise ranges like any
// input that does not fit
constexpr u64 kMaxRangeRecords = 0xffffffffull;   // sdbg_build's sort with payloads
u64 range_capacity(u64 avail, u32 W) {
    u64 lo = 0, hi = std::min<u64>(avail / (16ull * W) + 1, W == 1 ? radix_max_records(1, false) : radix_max_records(1, true));
    while (lo < hi) {
        u64 mid = lo + (hi - lo + 1) / 2;
        if (range_need(mid, W) <= avail) lo = mid; else hi = mid - 1;
    }
    return lo;
}

}  // namespace

extern "C" {

const char *sdbg_strerror(int status) {
    switch (status) {
        case SDBG_OK: return "ok";
        case SDBG_E_INVAL: return "invalid argument";
        case SDBG_E_BADBASE: return "read contains a character outside ACGTacgt";
        case SDBG_E_CAPACITY: return "output capacity too small";
        case SDBG_E_WORKSPACE: return "workspace too small";
        case SDBG_E_CUDA: return "CUDA error";
        case SDBG_E_UNSUPPORTED: return "unsupported k (must be in [1, 127])";
    }
    return "unknown status";
}

const char *sdbg_last_error(const sdbg_ctx *ctx) { return ctx ? ctx->err.c_str() : ""; }

int sdbg_ctx_create(sdbg_ctx **out, int device, void *cuda_stream, void *workspace, uint64_t workspace_bytes) {
    if (!out) return SDBG_E_INVAL;
    *out = nullptr;
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & (kAlign - 1))) return SDBG_E_INVAL;
    if (workspace_bytes < sdbg_min_workspace()) return SDBG_E_WORKSPACE;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { cudaGetLastError(); return SDBG_E_CUDA; }
    if (cudaSetDevice(device) != cudaSuccess) return SDBG_E_CUDA;
    {
        int sms = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) == cudaSuccess && sms > 0) g_num_sms = sms;
    }
    if (radix_setup() != 0) { cudaGetLastError(); return SDBG_E_CUDA; }
    if (hash_setup() != 0) { cudaGetLastError(); return SDBG_E_CUDA; }
    if (extract_scatter_setup() != 0) { cudaGetLastError(); return SDBG_E_CUDA; }
    sdbg_ctx *c = new sdbg_ctx();
    if (cudaHostAlloc(reinterpret_cast<void **>(&c->fetch_buf), kFetchBytes, cudaHostAllocMapped) != cudaSuccess) { cudaGetLastError(); delete c; return SDBG_E_CUDA; }
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    c->ws = (char *)workspace;
    c->ws_bytes = workspace_bytes;
    *out = c;
    return SDBG_OK;
}

void sdbg_ctx_destroy(sdbg_ctx *ctx) {
    if (!ctx) return;
    for (auto &p : ctx->pending) { cudaEventDestroy(p.a); cudaEventDestroy(p.b); }
    for (auto e : ctx->free_events) cudaEventDestroy(e);
    if (ctx->fetch_buf) cudaFreeHost(ctx->fetch_buf);
    delete ctx;
}

int sdbg_ctx_set_option(sdbg_ctx *ctx, int option, int value) {
    if (!ctx) return SDBG_E_INVAL;
    switch (option) {
        case SDBG_OPT_FORCE_WIDE: ctx->force_wide = value != 0; return SDBG_OK;
        case SDBG_OPT_STABLE_FIRST_PASS: ctx->no_unstable = value != 0; return SDBG_OK;
        case SDBG_OPT_NO_TABLE_COUNT: ctx->no_hash = value != 0; return SDBG_OK;
        case SDBG_OPT_NO_FUSED_EXTRACT: ctx->no_fused = value != 0; return SDBG_OK;
        case SDBG_OPT_WEAK_FINGERPRINT: ctx->weak_fp = value != 0; return SDBG_OK;
    }
    return ctx->fail(SDBG_E_INVAL, "unknown option");
}

int sdbg_ctx_set_timing(sdbg_ctx *ctx, int on) {
    if (!ctx) return SDBG_E_INVAL;
    ctx->timing = on != 0;
    return SDBG_OK;
}

int sdbg_ctx_get_timing(sdbg_ctx *ctx, sdbg_timing *out) {
    if (!ctx || !out) return SDBG_E_INVAL;
    CU(cudaStreamSynchronize(ctx->stream));
    for (auto &p : ctx->pending) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, p.a, p.b) == cudaSuccess) ctx->acc.ms[p.cls] += ms;
        ctx->free_events.push_back(p.a);
        ctx->free_events.push_back(p.b);
    }
    ctx->pending.clear();
    *out = ctx->acc;
    ctx->acc = sdbg_timing{};
    return SDBG_OK;
}

uint64_t sdbg_unstable_radix_launches(void) { return radix_unstable_launches(); }

uint32_t sdbg_key_words(uint32_t k) { return (2 * (k + 1) + 63) / 64; }

uint64_t sdbg_read_slots(uint64_t n_bases, uint64_t n_calls) {
    return (n_bases + 64 * std::max<u64>(n_calls, 1) + 63) / 64 * 64 + SDBG_READ_GUARD_SLOTS;
}

uint64_t sdbg_min_workspace(void) { return kFixedBytes + range_need(1ull << 16, 4); }

uint64_t sdbg_full_workspace(uint64_t n_bases, uint32_t k) {
    if (k < 1 || k > SDBG_MAX_K) return 0;
    const u64 need = kFixedBytes + range_need(2 * n_bases, sdbg_key_words(k)) + 4096;
    return std::max<u64>(need, sdbg_min_workspace());
}

uint64_t sdbg_workspace_for_records(uint64_t n_records, uint32_t k) {
    if (k < 1 || k > SDBG_MAX_K) return 0;
    const u64 need = kFixedBytes + range_need(n_records, sdbg_key_words(k)) + 4096;
    return std::max<u64>(need, sdbg_min_workspace());
}

int64_t sdbg_plan_ranges(const uint64_t *hist, uint64_t capacity, uint64_t *ranges, uint64_t max_ranges) {
    if (!hist || !ranges) return SDBG_E_INVAL;
    u64 nr = 0, lo = 0, sum = 0;
    for (u64 b = 0; b < SDBG_NUM_BUCKETS; ++b) {
        if (hist[b] > capacity) return SDBG_E_WORKSPACE;
        if (sum + hist[b] > capacity) {   // close [lo, b)
            if (nr == max_ranges) return SDBG_E_CAPACITY;
            ranges[3 * nr] = lo; ranges[3 * nr + 1] = b; ranges[3 * nr + 2] = sum; ++nr;
            lo = b; sum = 0;
        }
        sum += hist[b];
    }
    if (nr == max_ranges) return SDBG_E_CAPACITY;
    ranges[3 * nr] = lo; ranges[3 * nr + 1] = SDBG_NUM_BUCKETS; ranges[3 * nr + 2] = sum; ++nr;
    return (int64_t)nr;
}

}  // extern "C"

#include "api_pack.inc"
#include "api_count.inc"
#include "api_build.inc"
#include "api_full.inc"
#include "api_index.inc"

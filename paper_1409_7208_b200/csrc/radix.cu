// radix.cu — step a3: the sorter. "the bottleneck is sorting a set of (k+1)-mers ... in reverse
// lexicographical order of their length-k prefixes" (§2 ¶2). With the key encoding of include/sdbg.h that
// order is the ascending unsigned order of a 2(k+1)-bit integer, so the sort is a least-significant-digit radix sort
// over the significant bits only: P = sum over words of ceil(sigbits/8) stable 8-bit passes.
//
// Each pass is ONE kernel in the onesweep style (the paper's CX1-derived GPU sorter, is prior art, not
// the blueprint): global digit histograms are known up front (fused into the extractor), a tile of keys is ranked
// in shared memory (per-warp digit histograms + warp match ranking, stable in tile order), the tile's digit
// counts are chained to its predecessors by decoupled look-back on 64-bit status words (counts can exceed 2^32:
// config 3 has 3.2e9 records, config 5 31.6e9), and keys are staged bin-sorted in shared memory so that every
// digit's run leaves the SM as one coalesced segment. Tiles are ordered by an atomic ticket, which guarantees that
// every predecessor a tile waits on is already resident (forward progress).
//
// HBM traffic per pass: read n*K + write n*K bytes (K = 8w) — the algorithmic 2nK of DESIGN.md "Byte model" — plus
// 2 KiB of look-back state per tile.
#include "kernels.cuh"

namespace sdbg {

#ifndef SDBG_HW_MATCH
#define SDBG_HW_MATCH 0
#endif

template <int W, bool HAS_VAL> struct RadixCfg;
// THREADS x KPT records per tile; keys are staged in shared memory (TILE * 8W bytes).
template <> struct RadixCfg<1, false> { static constexpr int THREADS = 512, KPT = 16, MINB = 2; };
template <> struct RadixCfg<2, false> { static constexpr int THREADS = 512, KPT = 8,  MINB = 2; };
template <> struct RadixCfg<3, false> { static constexpr int THREADS = 512, KPT = 5,  MINB = 2; };
template <> struct RadixCfg<4, false> { static constexpr int THREADS = 512, KPT = 4,  MINB = 2; };
template <> struct RadixCfg<1, true>  { static constexpr int THREADS = 512, KPT = 10, MINB = 2; };
template <> struct RadixCfg<2, true>  { static constexpr int THREADS = 512, KPT = 6,  MINB = 2; };
template <> struct RadixCfg<3, true>  { static constexpr int THREADS = 512, KPT = 4,  MINB = 2; };
template <> struct RadixCfg<4, true>  { static constexpr int THREADS = 512, KPT = 3,  MINB = 2; };

constexpr u64 kValMask = (1ull << 54) - 1;

template <int W>
__device__ __forceinline__ u32 digit_of(const u64 (&key)[W], const PassDesc pd) {
    u64 kw = key[0];
#pragma unroll
    for (int j = 1; j < W; ++j) if (pd.word == j) kw = key[j];
    return (u32)(kw >> pd.shift) & ((1u << pd.bits) - 1u);
}

// lanes of the warp whose 8-bit digit equals mine
__device__ __forceinline__ u32 match_digit(u32 d) {
#if SDBG_HW_MATCH
    return __match_any_sync(0xffffffffu, d);
#else
    u32 m = 0xffffffffu;
#pragma unroll
    for (int b = 0; b < kRadixBits; ++b) {
        const bool bit = (d >> b) & 1u;
        const u32 bal = __ballot_sync(0xffffffffu, bit);
        m &= bit ? bal : ~bal;
    }
    return m;
#endif
}

template <int W, bool HAS_VAL>
__global__ void __launch_bounds__(RadixCfg<W, HAS_VAL>::THREADS, RadixCfg<W, HAS_VAL>::MINB)
onesweep_kernel(RadixArgs a) {
    using Cfg = RadixCfg<W, HAS_VAL>;
    constexpr int THREADS = Cfg::THREADS, KPT = Cfg::KPT, WARPS = THREADS / 32, TILE = THREADS * KPT;
    static_assert(THREADS >= kRadix, "one thread per bin");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    u64 *s_keys = reinterpret_cast<u64 *>(smem_raw);                 // W planes of TILE
    u64 *s_binout = s_keys + (size_t)TILE * W;                       // [256] global base - tile bin start
    u32 *s_whist = reinterpret_cast<u32 *>(s_binout + kRadix);       // [WARPS][256]
    u32 *s_binstart = s_whist + WARPS * kRadix;                      // [256]
    u32 *s_vals = s_binstart + kRadix;                               // [TILE] if HAS_VAL
    __shared__ u32 s_tile;
    __shared__ u32 s_wtot[kRadix / 32];

    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const u32 lt = lanemask_lt();
    const PassDesc pd = a.pass;

    if (tid == 0) s_tile = atomicAdd(a.ticket, 1u);
#pragma unroll
    for (int i = tid; i < WARPS * kRadix; i += THREADS) s_whist[i] = 0;
    __syncthreads();
    const u32 tile = s_tile;
    const u64 tile_base = (u64)tile * TILE;
    const u32 cnt = (a.n - tile_base < (u64)TILE) ? (u32)(a.n - tile_base) : (u32)TILE;

    // ---- load (warp-striped: lane l, step j -> tile index warp*32*KPT + j*32 + l) --------------------
    u64 key[KPT][W];
    u32 val[HAS_VAL ? KPT : 1];
    const u32 wbase = warp * 32u * KPT + lane;
#pragma unroll
    for (int j = 0; j < KPT; ++j) {
        const u32 ti = wbase + j * 32u;
        if (ti < cnt) {
            const u64 *src = a.keys_in + (tile_base + ti) * W;
            if constexpr (W == 1) {
                key[j][0] = ld_stream(src);
            } else if constexpr (W == 2) {
                ulonglong2 v = *reinterpret_cast<const ulonglong2 *>(src);
                key[j][0] = v.x; key[j][1] = v.y;
            } else if constexpr (W == 4) {
                ulonglong2 v0 = *reinterpret_cast<const ulonglong2 *>(src), v1 = *reinterpret_cast<const ulonglong2 *>(src + 2);
                key[j][0] = v0.x; key[j][1] = v0.y; key[j][2] = v1.x; key[j][3] = v1.y;
            } else {
#pragma unroll
                for (int q = 0; q < W; ++q) key[j][q] = src[q];
            }
            if constexpr (HAS_VAL) val[j] = a.vals_in[tile_base + ti];
        } else {
#pragma unroll
            for (int q = 0; q < W; ++q) key[j][q] = ~0ull;   // pads rank last in the last bin
            if constexpr (HAS_VAL) val[j] = 0;
        }
    }

    // ---- rank within the warp (stable in tile order) ---------------------------------------------------
    u32 *wh = s_whist + warp * kRadix;
    u32 rank2[(KPT + 1) / 2];   // two 16-bit ranks per register
#pragma unroll
    for (int j = 0; j < KPT; ++j) {
        const u32 d = digit_of<W>(key[j], pd);
        const u32 m = match_digit(d);
        const u32 leader = 31u - __clz(m);
        u32 prev = 0;
        if (lane == leader) { prev = wh[d]; wh[d] = prev + __popc(m); }
        prev = __shfl_sync(0xffffffffu, prev, leader);
        const u32 r = prev + __popc(m & lt);
        if (j & 1) rank2[j >> 1] |= r << 16; else rank2[j >> 1] = r;
        __syncwarp();
    }
    __syncthreads();

    // ---- per-bin: scan over warps, publish the tile count, look back ------------------------------------
    u32 my_cnt = 0, incl = 0;
    if (tid < kRadix) {
        u32 run = 0;
#pragma unroll
        for (int w = 0; w < WARPS; ++w) {
            const u32 t = s_whist[w * kRadix + tid];
            s_whist[w * kRadix + tid] = run;
            run += t;
        }
        my_cnt = run;   // includes pads (all in the last bin of this pass)
        incl = warp_incl_scan_add(my_cnt);
        if (lane == 31) s_wtot[warp] = incl;
    }
    __syncthreads();
    if (tid < kRadix) {
        u32 off = 0;
#pragma unroll
        for (int w = 0; w < kRadix / 32; ++w) off += (w < (int)warp) ? s_wtot[w] : 0u;
        const u32 bin_start = off + incl - my_cnt;
        s_binstart[tid] = bin_start;
        u32 real_cnt = my_cnt;
        if (tid == (1u << pd.bits) - 1u) real_cnt -= (u32)TILE - cnt;
        const u64 tagL = ((kStLocal << 8) | a.epoch), tagG = ((kStGlobal << 8) | a.epoch);
        u64 *lb = a.lookback + tid;
        u64 excl = 0;
        if (tile == 0) {
            st_relaxed(lb, (tagG << 54) | real_cnt);
        } else {
            st_relaxed(lb + (u64)tile * kRadix, (tagL << 54) | real_cnt);
            for (long long t = (long long)tile - 1; t >= 0; --t) {
                u64 v;
                do { v = ld_relaxed(lb + (u64)t * kRadix); } while ((v >> 54) != tagL && (v >> 54) != tagG);
                excl += v & kValMask;
                if ((v >> 54) == tagG) break;
            }
            st_relaxed(lb + (u64)tile * kRadix, (tagG << 54) | (excl + real_cnt));
        }
        s_binout[tid] = a.bin_base[tid] + excl - bin_start;
    }
    __syncthreads();

    // ---- scatter to shared memory in bin-sorted order ------------------------------------------------------
#pragma unroll
    for (int j = 0; j < KPT; ++j) {
        const u32 d = digit_of<W>(key[j], pd);
        const u32 r = (j & 1) ? (rank2[j >> 1] >> 16) : (rank2[j >> 1] & 0xffffu);
        const u32 pos = s_binstart[d] + wh[d] + r;
#pragma unroll
        for (int q = 0; q < W; ++q) s_keys[q * TILE + pos] = key[j][q];
        if constexpr (HAS_VAL) s_vals[pos] = val[j];
    }
    __syncthreads();

    // ---- coalesced write-out: position p of the tile goes to bin_out[digit] + p --------------------------------
#pragma unroll
    for (int i = 0; i < KPT; ++i) {
        const u32 p = i * THREADS + tid;
        if (p < cnt) {
            u64 kk[W];
#pragma unroll
            for (int q = 0; q < W; ++q) kk[q] = s_keys[q * TILE + p];
            const u32 d = digit_of<W>(kk, pd);
            const u64 dst = s_binout[d] + p;
            u64 *o = a.keys_out + dst * W;
            if constexpr (W == 1) {
                o[0] = kk[0];
            } else if constexpr (W == 2) {
                *reinterpret_cast<ulonglong2 *>(o) = make_ulonglong2(kk[0], kk[1]);
            } else if constexpr (W == 4) {
                *reinterpret_cast<ulonglong2 *>(o) = make_ulonglong2(kk[0], kk[1]);
                *reinterpret_cast<ulonglong2 *>(o + 2) = make_ulonglong2(kk[2], kk[3]);
            } else {
#pragma unroll
                for (int q = 0; q < W; ++q) o[q] = kk[q];
            }
            if constexpr (HAS_VAL) a.vals_out[dst] = s_vals[p];
        }
    }
}

template <int W, bool HAS_VAL>
static constexpr size_t radix_smem_bytes() {
    using Cfg = RadixCfg<W, HAS_VAL>;
    constexpr size_t TILE = (size_t)Cfg::THREADS * Cfg::KPT, WARPS = Cfg::THREADS / 32;
    return TILE * W * 8 + kRadix * 8 + WARPS * kRadix * 4 + kRadix * 4 + (HAS_VAL ? TILE * 4 : 0);
}

template <int W, bool HAS_VAL>
static int setup_one() {
    return (int)cudaFuncSetAttribute(onesweep_kernel<W, HAS_VAL>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)radix_smem_bytes<W, HAS_VAL>());
}

int radix_setup() {
    int e = 0;
    if ((e = setup_one<1, false>())) return e;
    if ((e = setup_one<2, false>())) return e;
    if ((e = setup_one<3, false>())) return e;
    if ((e = setup_one<4, false>())) return e;
    if ((e = setup_one<1, true>())) return e;
    if ((e = setup_one<2, true>())) return e;
    if ((e = setup_one<3, true>())) return e;
    if ((e = setup_one<4, true>())) return e;
    return 0;
}

template <int W, bool HAS_VAL>
static constexpr u64 tile_of() { return (u64)RadixCfg<W, HAS_VAL>::THREADS * RadixCfg<W, HAS_VAL>::KPT; }

u64 radix_tile_records(u32 W, bool v) {
    switch (W) {
        case 1: return v ? tile_of<1, true>() : tile_of<1, false>();
        case 2: return v ? tile_of<2, true>() : tile_of<2, false>();
        case 3: return v ? tile_of<3, true>() : tile_of<3, false>();
        case 4: return v ? tile_of<4, true>() : tile_of<4, false>();
    }
    return 0;
}

template <int W, bool HAS_VAL>
static int launch_one(const RadixArgs &a, cudaStream_t s) {
    const u64 tiles = (a.n + tile_of<W, HAS_VAL>() - 1) / tile_of<W, HAS_VAL>();
    if (tiles == 0) return 0;
    if (tiles > 0x7fffffffull) return (int)cudaErrorInvalidValue;
    onesweep_kernel<W, HAS_VAL><<<(unsigned)tiles, RadixCfg<W, HAS_VAL>::THREADS, radix_smem_bytes<W, HAS_VAL>(), s>>>(a);
    return (int)cudaGetLastError();
}

int launch_radix_pass(const RadixArgs &a, cudaStream_t s) {
    const bool v = a.vals_in != nullptr;
    switch (a.W) {
        case 1: return v ? launch_one<1, true>(a, s) : launch_one<1, false>(a, s);
        case 2: return v ? launch_one<2, true>(a, s) : launch_one<2, false>(a, s);
        case 3: return v ? launch_one<3, true>(a, s) : launch_one<3, false>(a, s);
        case 4: return v ? launch_one<4, true>(a, s) : launch_one<4, false>(a, s);
    }
    return (int)cudaErrorInvalidValue;
}

// ---- histogram helpers ------------------------------------------------------------------------------------------

// in-place exclusive scan of each pass's 256 u64 bins; one block per pass
__global__ void __launch_bounds__(kRadix) scan_hist_kernel(u64 *hist) {
    __shared__ u64 s_w[kRadix / 32];
    u64 *h = hist + (size_t)blockIdx.x * kRadix;
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const u64 v = h[tid];
    u64 incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        u64 t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= (u32)o) incl += t;
    }
    if (lane == 31) s_w[warp] = incl;
    __syncthreads();
    u64 off = 0;
    for (u32 w = 0; w < warp; ++w) off += s_w[w];
    h[tid] = off + incl - v;
}

void launch_scan_hist(u64 *digit_hist, int n_passes, cudaStream_t s) {
    if (n_passes > 0) scan_hist_kernel<<<n_passes, kRadix, 0, s>>>(digit_hist);
}

// digit histograms of all passes over an existing key array (sdbg_build's unsorted path)
template <int W>
__global__ void __launch_bounds__(256) key_hist_kernel(const u64 *__restrict__ keys, u64 n, PassTable pt, u64 *hist) {
    extern __shared__ u32 s_hist[];
    for (int i = threadIdx.x; i < pt.n * kRadix; i += blockDim.x) s_hist[i] = 0;
    __syncthreads();
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (u64)gridDim.x * blockDim.x) {
        u64 key[W];
#pragma unroll
        for (int q = 0; q < W; ++q) key[q] = keys[i * W + q];
        for (int p = 0; p < pt.n; ++p) atomicAdd(&s_hist[p * kRadix + digit_of<W>(key, pt.p[p])], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < pt.n * kRadix; i += blockDim.x)
        if (s_hist[i]) atomicAdd(&hist[i], (u64)s_hist[i]);
}

void launch_key_hist(const u64 *keys, u64 n, u32 W, const PassTable &pt, u64 *hist, cudaStream_t s) {
    if (n == 0) return;
    u64 blocks = (n + 255) / 256;
    if (blocks > (u64)kNumSMs * 8) blocks = (u64)kNumSMs * 8;
    size_t smem = (size_t)pt.n * kRadix * 4;
    switch (W) {
        case 1: key_hist_kernel<1><<<(unsigned)blocks, 256, smem, s>>>(keys, n, pt, hist); break;
        case 2: key_hist_kernel<2><<<(unsigned)blocks, 256, smem, s>>>(keys, n, pt, hist); break;
        case 3: key_hist_kernel<3><<<(unsigned)blocks, 256, smem, s>>>(keys, n, pt, hist); break;
        case 4: key_hist_kernel<4><<<(unsigned)blocks, 256, smem, s>>>(keys, n, pt, hist); break;
    }
}

}  // namespace sdbg

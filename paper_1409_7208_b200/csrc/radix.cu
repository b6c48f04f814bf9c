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

#ifndef SDBG_LB_SKIP
#define SDBG_LB_SKIP 0   // timing experiments only: wrong results
#endif
#ifndef SDBG_LB_DEPTH
#define SDBG_LB_DEPTH 4  // independent look-back loads in flight per bin
#endif
#ifndef SDBG_MERGE_BINSTART
#define SDBG_MERGE_BINSTART 1
#endif
#ifndef SDBG_FULL_SPEC
#define SDBG_FULL_SPEC 0   // duplicating the load/store loops for full tiles overflows the instruction cache: slower
#endif
#ifndef SDBG_VSPLIT
#define SDBG_VSPLIT 1    // independent ranking chains ("virtual warps") per warp
#endif

template <int W, bool HAS_VAL> struct RadixCfg;
// THREADS x KPT records per tile; keys are staged in shared memory (TILE * 8W bytes).
#ifndef SDBG_R1_THREADS
#define SDBG_R1_THREADS 512
#define SDBG_R1_KPT 16
#define SDBG_R1_MINB 2
#endif
template <> struct RadixCfg<1, false> { static constexpr int THREADS = SDBG_R1_THREADS, KPT = SDBG_R1_KPT, MINB = SDBG_R1_MINB; };
template <> struct RadixCfg<2, false> { static constexpr int THREADS = 512, KPT = 8,  MINB = 2; };
template <> struct RadixCfg<3, false> { static constexpr int THREADS = 512, KPT = 5,  MINB = 2; };
template <> struct RadixCfg<4, false> { static constexpr int THREADS = 512, KPT = 4,  MINB = 2; };
template <> struct RadixCfg<1, true>  { static constexpr int THREADS = 512, KPT = 10, MINB = 2; };
template <> struct RadixCfg<2, true>  { static constexpr int THREADS = 512, KPT = 6,  MINB = 2; };
template <> struct RadixCfg<3, true>  { static constexpr int THREADS = 512, KPT = 4,  MINB = 2; };
template <> struct RadixCfg<4, true>  { static constexpr int THREADS = 512, KPT = 3,  MINB = 2; };

constexpr u64 kValMask = (1ull << 54) - 1;
constexpr int kVSplit = SDBG_VSPLIT;

template <int W>
__device__ __forceinline__ u32 digit_of(const u64 (&key)[W], const PassDesc pd) {
    u64 kw = key[0];
#pragma unroll
    for (int j = 1; j < W; ++j) if (pd.word == j) kw = key[j];
    return (u32)(kw >> pd.shift) & ((1u << pd.bits) - 1u);
}

// lanes of the warp whose 8-bit digit equals mine: 8 ballots, 4 SASS instructions per bit
// (LOP3 -> predicate, VOTE, predicated NOT, AND) — the hardware match.any is ~3x slower on sm_100.
__device__ __forceinline__ u32 match_digit(u32 d) {
    u32 m = 0xffffffffu;
#pragma unroll
    for (int b = 0; b < kRadixBits; ++b) {
        asm("{\n\t.reg .pred p;\n\t.reg .b32 t, bal;\n\t"
            "and.b32 t, %1, %2;\n\tsetp.ne.u32 p, t, 0;\n\t"
            "vote.sync.ballot.b32 bal, p, 0xffffffff;\n\t"
            "@!p not.b32 bal, bal;\n\t"
            "and.b32 %0, %0, bal;\n\t}" : "+r"(m) : "r"(d), "r"(1u << b));
    }
    return m;
}

template <int W>
__device__ __forceinline__ void load_rec(const u64 *__restrict__ src, u64 (&k)[W]) {
    if constexpr (W == 1) {
        k[0] = ld_stream(src);
    } else if constexpr (W == 2) {
        ulonglong2 v = *reinterpret_cast<const ulonglong2 *>(src);
        k[0] = v.x; k[1] = v.y;
    } else if constexpr (W == 4) {
        ulonglong2 v0 = *reinterpret_cast<const ulonglong2 *>(src), v1 = *reinterpret_cast<const ulonglong2 *>(src + 2);
        k[0] = v0.x; k[1] = v0.y; k[2] = v1.x; k[3] = v1.y;
    } else {
#pragma unroll
        for (int q = 0; q < W; ++q) k[q] = src[q];
    }
}
template <int W>
__device__ __forceinline__ void store_rec(u64 *__restrict__ o, const u64 (&k)[W]) {
    if constexpr (W == 1) {
        o[0] = k[0];
    } else if constexpr (W == 2) {
        *reinterpret_cast<ulonglong2 *>(o) = make_ulonglong2(k[0], k[1]);
    } else if constexpr (W == 4) {
        *reinterpret_cast<ulonglong2 *>(o) = make_ulonglong2(k[0], k[1]);
        *reinterpret_cast<ulonglong2 *>(o + 2) = make_ulonglong2(k[2], k[3]);
    } else {
#pragma unroll
        for (int q = 0; q < W; ++q) o[q] = k[q];
    }
}

template <int W, bool HAS_VAL>
__global__ void __launch_bounds__(RadixCfg<W, HAS_VAL>::THREADS, RadixCfg<W, HAS_VAL>::MINB)
onesweep_kernel(RadixArgs a) {
    using Cfg = RadixCfg<W, HAS_VAL>;
    constexpr int THREADS = Cfg::THREADS, KPT = Cfg::KPT, WARPS = THREADS / 32, TILE = THREADS * KPT;
    constexpr int VS = (KPT >= 2 * kVSplit) ? kVSplit : 1;      // ranking chains per warp
    constexpr int VW = WARPS * VS;                              // virtual warps
    constexpr int H = (KPT + VS - 1) / VS;                      // steps per chain
    static_assert(THREADS >= kRadix, "one thread per bin");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    u64 *s_keys = reinterpret_cast<u64 *>(smem_raw);                 // W planes of TILE
    u64 *s_binout = s_keys + (size_t)TILE * W;                       // [256] global base - tile bin start
    u32 *s_whist = reinterpret_cast<u32 *>(s_binout + kRadix);       // [VW][256]: count, then tile position of the group
    u32 *s_vals = s_whist + VW * kRadix;                             // [TILE] if HAS_VAL
    __shared__ u32 s_tile;
    __shared__ u32 s_wtot[kRadix / 32];
#if !SDBG_MERGE_BINSTART
    __shared__ u32 s_binstart[kRadix];
#endif

    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const u32 lt = lanemask_lt();
    const PassDesc pd = a.pass;

    if (tid == 0) s_tile = atomicAdd(a.ticket, 1u);
#pragma unroll
    for (int i = tid; i < VW * kRadix; i += THREADS) s_whist[i] = 0;
    __syncthreads();
    const u32 tile = s_tile;
    const u64 tile_base = (u64)tile * TILE;
    const u32 cnt = (a.n - tile_base < (u64)TILE) ? (u32)(a.n - tile_base) : (u32)TILE;
    const bool full = SDBG_FULL_SPEC && cnt == (u32)TILE;

    // ---- load (warp-striped: lane l, step j -> tile index warp*32*KPT + j*32 + l) --------------------
    u64 key[KPT][W];
    u32 val[HAS_VAL ? KPT : 1];
    const u32 wbase = warp * 32u * KPT + lane;
    if (full) {
#pragma unroll
        for (int j = 0; j < KPT; ++j) {
            load_rec<W>(a.keys_in + (tile_base + wbase + j * 32u) * W, key[j]);
            if constexpr (HAS_VAL) val[j] = a.vals_in[tile_base + wbase + j * 32u];
        }
    } else {
#pragma unroll
        for (int j = 0; j < KPT; ++j) {
            const u32 ti = wbase + j * 32u;
            if (ti < cnt) {
                load_rec<W>(a.keys_in + (tile_base + ti) * W, key[j]);
                if constexpr (HAS_VAL) val[j] = a.vals_in[tile_base + ti];
            } else {
#pragma unroll
                for (int q = 0; q < W; ++q) key[j][q] = ~0ull;   // pads rank last in the last bin
                if constexpr (HAS_VAL) val[j] = 0;
            }
        }
    }

    // ---- rank within the (virtual) warp, stable in tile order ---------------------------------------------
    // Chain c of the warp owns steps [c*H, (c+1)*H): VS independent smem dependency chains per warp.
    u32 rank2[(KPT + 1) / 2];   // two 16-bit ranks per register
#pragma unroll
    for (int i = 0; i < (KPT + 1) / 2; ++i) rank2[i] = 0;
#pragma unroll
    for (int jj = 0; jj < H; ++jj) {
#pragma unroll
        for (int c = 0; c < VS; ++c) {
            const int j = c * H + jj;
            if (j < KPT) {
                u32 *wh = s_whist + (warp * VS + c) * kRadix;
                const u32 d = digit_of<W>(key[j], pd);
                const u32 m = match_digit(d);
                const u32 prev = wh[d];                            // same address within the group: broadcast read
                __syncwarp();
                if ((m >> lane) <= 1u) wh[d] = prev + __popc(m);   // highest lane of the group updates the count
                const u32 r = prev + __popc(m & lt);
                rank2[j >> 1] |= (j & 1) ? (r << 16) : r;
            }
        }
        __syncwarp();
    }
    __syncthreads();

    // ---- per bin: totals over the virtual warps, publish the tile's count (LOCAL) as early as possible ------------
    u32 my_cnt = 0, incl = 0, real_cnt = 0;
    const u64 tagL = ((kStLocal << 8) | a.epoch), tagG = ((kStGlobal << 8) | a.epoch);
    u64 *lb = a.lookback + tid;
    if (tid < kRadix) {
#if SDBG_MERGE_BINSTART
#pragma unroll
        for (int v = 0; v < VW; ++v) my_cnt += s_whist[v * kRadix + tid];
#else
#pragma unroll
        for (int v = 0; v < VW; ++v) {
            const u32 t = s_whist[v * kRadix + tid];
            s_whist[v * kRadix + tid] = my_cnt;
            my_cnt += t;
        }
#endif
        real_cnt = my_cnt;                                            // my_cnt includes the pads (last bin of the pass)
        if (tid == (1u << pd.bits) - 1u) real_cnt -= (u32)TILE - cnt;
        st_relaxed(lb + (u64)tile * kRadix, ((tile == 0 ? tagG : tagL) << 54) | real_cnt);
        incl = warp_incl_scan_add(my_cnt);
        if (lane == 31) s_wtot[warp] = incl;
    }
    __syncthreads();
    u32 bin_start = 0;
    if (tid < kRadix) {
        u32 off = 0;
#pragma unroll
        for (int w = 0; w < kRadix / 32; ++w) off += (w < (int)warp) ? s_wtot[w] : 0u;
        bin_start = off + incl - my_cnt;
#if SDBG_MERGE_BINSTART
        // entry (v, bin) becomes the tile position of the first key of digit `bin` held by virtual warp v
        u32 run = bin_start;
#pragma unroll
        for (int v = 0; v < VW; ++v) {
            const u32 t = s_whist[v * kRadix + tid];
            s_whist[v * kRadix + tid] = run;
            run += t;
        }
#else
        s_binstart[tid] = bin_start;
#endif
    }
    __syncthreads();

    // ---- scatter to shared memory in bin-sorted order ------------------------------------------------------
#pragma unroll
    for (int j = 0; j < KPT; ++j) {
        const u32 d = digit_of<W>(key[j], pd);
        const u32 r = (j & 1) ? (rank2[j >> 1] >> 16) : (rank2[j >> 1] & 0xffffu);
#if SDBG_MERGE_BINSTART
        const u32 pos = s_whist[(warp * VS + j / H) * kRadix + d] + r;
#else
        const u32 pos = s_binstart[d] + s_whist[(warp * VS + j / H) * kRadix + d] + r;
#endif
#pragma unroll
        for (int q = 0; q < W; ++q) s_keys[q * TILE + pos] = key[j][q];
        if constexpr (HAS_VAL) s_vals[pos] = val[j];
    }

    // ---- decoupled look-back (one thread per bin), after the scatter so that predecessors had time to finish ---
    if (tid < kRadix) {
        u64 excl = 0;
        if (tile != 0 && !SDBG_LB_SKIP) {
            // walk back in batches of SDBG_LB_DEPTH independent loads (the chain of dependent L2 round trips is
            // the cost of the look-back); entries not ready yet are re-polled one by one
            long long t = (long long)tile - 1;
            bool done = false;
            while (!done) {
                u64 v[SDBG_LB_DEPTH];
#pragma unroll
                for (int q = 0; q < SDBG_LB_DEPTH; ++q) v[q] = (t - q >= 0) ? ld_relaxed(lb + (u64)(t - q) * kRadix) : (tagG << 54);
#pragma unroll
                for (int q = 0; q < SDBG_LB_DEPTH; ++q) {
                    if (!done) {
                        u64 x = v[q];
                        while ((x >> 54) != tagL && (x >> 54) != tagG) x = ld_relaxed(lb + (u64)(t - q) * kRadix);
                        excl += x & kValMask;
                        done = (x >> 54) == tagG;
                    }
                }
                t -= SDBG_LB_DEPTH;
            }
            st_relaxed(lb + (u64)tile * kRadix, (tagG << 54) | (excl + real_cnt));
        }
        s_binout[tid] = a.bin_base[tid] + excl - bin_start;
    }
    __syncthreads();

    // ---- coalesced write-out: position p of the tile goes to bin_out[digit] + p --------------------------------
    if (full) {
#pragma unroll
        for (int i = 0; i < KPT; ++i) {
            const u32 p = i * THREADS + tid;
            u64 kk[W];
#pragma unroll
            for (int q = 0; q < W; ++q) kk[q] = s_keys[q * TILE + p];
            const u64 dst = s_binout[digit_of<W>(kk, pd)] + p;
            store_rec<W>(a.keys_out + dst * W, kk);
            if constexpr (HAS_VAL) a.vals_out[dst] = s_vals[p];
        }
    } else {
#pragma unroll
        for (int i = 0; i < KPT; ++i) {
            const u32 p = i * THREADS + tid;
            if (p < cnt) {
                u64 kk[W];
#pragma unroll
                for (int q = 0; q < W; ++q) kk[q] = s_keys[q * TILE + p];
                const u64 dst = s_binout[digit_of<W>(kk, pd)] + p;
                store_rec<W>(a.keys_out + dst * W, kk);
                if constexpr (HAS_VAL) a.vals_out[dst] = s_vals[p];
            }
        }
    }
}

template <int W, bool HAS_VAL>
static constexpr size_t radix_smem_bytes() {
    using Cfg = RadixCfg<W, HAS_VAL>;
    constexpr size_t TILE = (size_t)Cfg::THREADS * Cfg::KPT, WARPS = Cfg::THREADS / 32;
    constexpr size_t VW = WARPS * ((Cfg::KPT >= 2 * kVSplit) ? kVSplit : 1);
    return TILE * W * 8 + kRadix * 8 + VW * kRadix * 4 + (HAS_VAL ? TILE * 4 : 0);
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

// count.cu — step a4: run-length counting of the sorted records and the solid filter:
// "all (k+1)-mers from the input reads are sorted and counted, and only (k+1)-mers that appear at least d (2 by
// default) times are kept" (§2 ¶3; cnt >= d, reading A8; counts saturate at 2^32-1, A9).
//
// One streaming pass. A record i is a run TAIL iff i == n-1 or key[i] != key[i+1]; the run ending at tail i has
// length (i+1) - (index+1 of the previous tail). Runs may span any number of tiles, so the "previous tail" is an
// exclusive max-scan and the output position an exclusive sum-scan, both chained across tiles by decoupled
// look-back (one warp inspects 32 predecessors at a time). Tiles are ordered by an atomic ticket.
//
// Also here: the merge kernels of sdbg_build's unsorted path (equal keys merged by summing mult).
#include "kernels.cuh"

namespace sdbg {

constexpr u64 kLbVal = (1ull << 62) - 1;

// Decoupled look-back over per-tile status words ([63:62] status, [61:0] value); called by all 32 lanes of ONE warp.
// Publishes this tile's aggregate, returns the exclusive prefix over tiles [0, tile), then publishes the inclusive one.
template <bool IS_MAX>
__device__ __forceinline__ u64 tile_lookback(u64 *state, u32 tile, u64 aggregate) {
    const u32 lane = lane_id();
    if (tile == 0) {
        if (lane == 0) st_relaxed(state, (kStGlobal << 62) | aggregate);
        return 0;
    }
    if (lane == 0) st_relaxed(state + tile, (kStLocal << 62) | aggregate);
    u64 excl = 0;
    long long pos = (long long)tile - 1;
    while (true) {
        const long long idx = pos - (long long)lane;
        u64 v = kStGlobal << 62;   // virtual tiles before the first: inclusive identity
        if (idx >= 0) {
            do { v = ld_relaxed(state + idx); } while ((v >> 62) == kStInvalid);
        }
        const u32 gm = __ballot_sync(0xffffffffu, (v >> 62) == kStGlobal);
        const u32 first = gm ? (u32)__ffs(gm) - 1u : 31u;
        u64 x = (lane <= first) ? (v & kLbVal) : 0ull;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const u64 y = __shfl_xor_sync(0xffffffffu, x, o);
            x = IS_MAX ? (x > y ? x : y) : (x + y);
        }
        excl = IS_MAX ? (excl > x ? excl : x) : (excl + x);
        if (gm) break;
        pos -= 32;
    }
    const u64 inc = IS_MAX ? (excl > aggregate ? excl : aggregate) : (excl + aggregate);
    if (lane == 0) st_relaxed(state + tile, (kStGlobal << 62) | inc);
    return excl;
}

// Block-wide exclusive scan of one u32 per thread (add or max; identity 0). All threads must call it.
template <int THREADS, bool IS_MAX>
__device__ __forceinline__ u32 block_excl_scan(u32 v, u32 *s_warp /*[THREADS/32]*/, u32 &total) {
    const u32 lane = lane_id(), warp = threadIdx.x >> 5;
    u32 incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const u32 t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= (u32)o) incl = IS_MAX ? max(incl, t) : incl + t;
    }
    u32 excl = __shfl_up_sync(0xffffffffu, incl, 1);
    if (lane == 0) excl = 0;
    __syncthreads();   // protect s_warp reuse
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    u32 off = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < THREADS / 32; ++w) {
        const u32 t = s_warp[w];
        if (w < (int)warp) off = IS_MAX ? max(off, t) : off + t;
        tot = IS_MAX ? max(tot, t) : tot + t;
    }
    total = tot;
    return IS_MAX ? max(off, excl) : off + excl;
}

template <int W>
__device__ __forceinline__ void load_key(const u64 *__restrict__ keys, u64 idx, u64 (&k)[W]) {
    const u64 *src = keys + idx * W;
    if constexpr (W == 2) {
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
__device__ __forceinline__ bool key_ne(const u64 (&a)[W], const u64 (&b)[W]) {
    bool ne = false;
#pragma unroll
    for (int q = 0; q < W; ++q) ne = ne || (a[q] != b[q]);
    return ne;
}

template <int W> struct CountCfg { static constexpr int THREADS = 512, IPT = (W == 1 ? 8 : W == 2 ? 4 : 2); };

template <int W>
__global__ void __launch_bounds__(CountCfg<W>::THREADS) count_filter_kernel(CountArgs a, DevState *st) {
    constexpr int THREADS = CountCfg<W>::THREADS, IPT = CountCfg<W>::IPT, TILE = THREADS * IPT;
    __shared__ u32 s_tile;
    __shared__ u32 s_warp[THREADS / 32];
    __shared__ u64 s_bcast[2];
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(a.ticket, 1u);
    __syncthreads();
    const u32 tile = s_tile;
    const u32 ntiles = (u32)((a.n + TILE - 1) / TILE);
    const u64 tile_base = (u64)tile * TILE;
    const u64 idx0 = tile_base + (u64)tid * IPT;
    const u64 out_base = st->out_cursor[a.range_parity];   // solid edges appended by earlier ranges (never written by this launch)

    // ---- load IPT consecutive records + the one after them -------------------------------------------------------
    u64 key[IPT + 1][W];
    if (idx0 + IPT + 1 <= a.n && W == 1) {
        // vector path: IPT*8 bytes are 16-byte aligned
#pragma unroll
        for (int j = 0; j < IPT; j += 2) {
            ulonglong2 v = *reinterpret_cast<const ulonglong2 *>(a.keys + idx0 + j);
            key[j][0] = v.x; key[j + 1][0] = v.y;
        }
        key[IPT][0] = a.keys[idx0 + IPT];
    } else {
#pragma unroll
        for (int j = 0; j <= IPT; ++j) {
            if (idx0 + j < a.n) load_key<W>(a.keys, idx0 + j, key[j]);
            else {
#pragma unroll
                for (int q = 0; q < W; ++q) key[j][q] = 0;
            }
        }
    }
    u32 tails = 0, last_local = 0;   // last_local: tile-relative index+1 of my last tail (0 = none)
#pragma unroll
    for (int j = 0; j < IPT; ++j) {
        const u64 idx = idx0 + j;
        const bool t = idx < a.n && (idx + 1 == a.n || key_ne<W>(key[j], key[j + 1]));
        if (t) { tails |= 1u << j; last_local = tid * IPT + j + 1; }
    }

    // ---- previous tail: exclusive max-scan in the block, look-back across tiles --------------------------------
    u32 tile_max;
    const u32 excl_max = block_excl_scan<THREADS, true>(last_local, s_warp, tile_max);
    if (warp == 0) {
        const u64 p = tile_lookback<true>(a.lookback, tile, tile_max ? tile_base + tile_max : 0ull);
        if (lane == 0) s_bcast[0] = p;
    }
    __syncthreads();
    u64 prev = excl_max ? tile_base + excl_max : s_bcast[0];   // index+1 of the last tail before my first record

    // ---- run lengths, solid flags, statistics --------------------------------------------------------------------
    u32 solid = 0, n_solid = 0;
    u64 len[IPT];
    u64 sum_mult = 0, csum = 0;
#pragma unroll
    for (int j = 0; j < IPT; ++j) {
        len[j] = 0;
        if ((tails >> j) & 1u) {
            const u64 e = idx0 + j + 1;
            len[j] = e - prev;
            prev = e;
            if (len[j] >= (u64)a.d) { solid |= 1u << j; ++n_solid; sum_mult += len[j]; }
            if (a.want_csum) csum += len[j] * mix_key<W>(key[j]);
        }
    }
    u32 tile_solid;
    const u32 excl_sum = block_excl_scan<THREADS, false>(n_solid, s_warp, tile_solid);
    if (warp == 0) {
        const u64 p = tile_lookback<false>(a.lookback + ntiles, tile, (u64)tile_solid);
        if (lane == 0) {
            s_bcast[1] = p;
            if (tile == ntiles - 1) st->out_cursor[a.range_parity ^ 1] = out_base + p + tile_solid;
        }
    }
    __syncthreads();
    u64 pos = out_base + s_bcast[1] + excl_sum;
#pragma unroll
    for (int j = 0; j < IPT; ++j) {
        if ((solid >> j) & 1u) {
            if (pos < a.out_cap) {
#pragma unroll
                for (int q = 0; q < W; ++q) a.out_keys[pos * W + q] = key[j][q];
                a.out_mult[pos] = len[j] > 0xffffffffull ? 0xffffffffu : (u32)len[j];
            }
            ++pos;
        }
    }
    // ---- statistics: one atomic per warp ------------------------------------------------------------------------------
    u64 nt = warp_reduce_add64((u64)__popc(tails));
    sum_mult = warp_reduce_add64(sum_mult);
    if (lane == 0) {
        if (nt) atomicAdd(&st->n_distinct, nt);
        if (sum_mult) atomicAdd(&st->sum_solid_mult, sum_mult);
    }
    if (a.want_csum) {
        csum = warp_reduce_add64(csum);
        if (lane == 0 && csum) atomicAdd(&st->csum_distinct, csum);
    }
}

template <int W> static constexpr u64 count_tile() { return (u64)CountCfg<W>::THREADS * CountCfg<W>::IPT; }

u64 count_tile_records(u32 W) {
    switch (W) { case 1: return count_tile<1>(); case 2: return count_tile<2>(); case 3: return count_tile<3>(); case 4: return count_tile<4>(); }
    return 0;
}

template <int W>
static int launch_count_w(const CountArgs &a, DevState *st, cudaStream_t s) {
    const u64 tiles = (a.n + count_tile<W>() - 1) / count_tile<W>();
    if (tiles == 0) return 0;
    if (tiles > 0x7fffffffull) return (int)cudaErrorInvalidValue;
    count_filter_kernel<W><<<(unsigned)tiles, CountCfg<W>::THREADS, 0, s>>>(a, st);
    return (int)cudaGetLastError();
}

int launch_count_filter(const CountArgs &a, DevState *st, cudaStream_t s) {
    switch (a.W) {
        case 1: return launch_count_w<1>(a, st, s);
        case 2: return launch_count_w<2>(a, st, s);
        case 3: return launch_count_w<3>(a, st, s);
        case 4: return launch_count_w<4>(a, st, s);
    }
    return (int)cudaErrorInvalidValue;
}

// ---- sdbg_build unsorted path: merge equal adjacent keys, summing mult ------------------------------------------------
// Pass 1: head flags -> distinct index of every record (inclusive sum-scan, look-back across tiles); heads write their
// key, every record adds its mult into acc[distinct index]. Pass 2: saturate acc into out_mult.
constexpr int kMergeThreads = 256;

template <int W>
__global__ void __launch_bounds__(kMergeThreads) merge_kernel(MergeArgs a, DevState *st) {
    __shared__ u32 s_tile;
    __shared__ u32 s_warp[kMergeThreads / 32];
    __shared__ u64 s_bcast;
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(a.ticket, 1u);
    __syncthreads();
    const u32 tile = s_tile;
    const u32 ntiles = (u32)((a.n + kMergeThreads - 1) / kMergeThreads);
    const u64 idx = (u64)tile * kMergeThreads + tid;
    u64 key[W], prevk[W];
    bool head = false;
    if (idx < a.n) {
        load_key<W>(a.keys, idx, key);
        if (idx == 0) head = true;
        else { load_key<W>(a.keys, idx - 1, prevk); head = key_ne<W>(key, prevk); }
    }
    u32 tile_heads;
    const u32 excl = block_excl_scan<kMergeThreads, false>(head ? 1u : 0u, s_warp, tile_heads);
    if (warp == 0) {
        const u64 p = tile_lookback<false>(a.lookback, tile, (u64)tile_heads);
        if (lane == 0) {
            s_bcast = p;
            if (tile == ntiles - 1) st->merge_heads = p + tile_heads;
        }
    }
    __syncthreads();
    if (idx < a.n) {
        const u64 di = s_bcast + excl + (head ? 1u : 0u) - 1u;   // distinct index of this record
        if (head) {
#pragma unroll
            for (int q = 0; q < W; ++q) a.out_keys[di * W + q] = key[q];
        }
        atomicAdd(&a.acc[di], (u64)a.mult[idx]);
    }
}

__global__ void __launch_bounds__(256) merge_finish_kernel(const u64 *acc, u32 *out_mult, u64 n, const DevState *st) {
    const u64 m = st->merge_heads;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < m && i < n; i += (u64)gridDim.x * blockDim.x)
        out_mult[i] = acc[i] > 0xffffffffull ? 0xffffffffu : (u32)acc[i];
}

u64 merge_tile_records() { return kMergeThreads; }

void launch_merge(const MergeArgs &a, DevState *st, cudaStream_t s) {
    if (a.n == 0) return;
    const u64 tiles = (a.n + kMergeThreads - 1) / kMergeThreads;
    switch (a.W) {
        case 1: merge_kernel<1><<<(unsigned)tiles, kMergeThreads, 0, s>>>(a, st); break;
        case 2: merge_kernel<2><<<(unsigned)tiles, kMergeThreads, 0, s>>>(a, st); break;
        case 3: merge_kernel<3><<<(unsigned)tiles, kMergeThreads, 0, s>>>(a, st); break;
        case 4: merge_kernel<4><<<(unsigned)tiles, kMergeThreads, 0, s>>>(a, st); break;
    }
    u64 blocks = (a.n + 255) / 256;
    if (blocks > (u64)kNumSMs * 8) blocks = (u64)kNumSMs * 8;
    merge_finish_kernel<<<(unsigned)blocks, 256, 0, s>>>(a.acc, a.out_mult, a.n, st);
}

}  // namespace sdbg

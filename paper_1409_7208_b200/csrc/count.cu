// count.cu — step a4: run-length counting of the sorted records and the solid filter:
// "all (k+1)-mers from the input reads are sorted and counted, and only (k+1)-mers that appear at least d (2 by
// default) times are kept" (§2 ¶3; cnt >= d, reading A8; counts saturate at 2^32-1, A9).
//
// One streaming sweep over the sorted records, a scan, and a short second kernel that copies the solid edges out from
// what the sweep has noted about them; see count_chunks_kernel and count_write_kernel.
//
// Also here: the merge kernels of sdbg_build's unsorted path (equal keys merged by summing mult).
#include "kernels.cuh"
#include <type_traits>

namespace sdbg {

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

template <int W>
__device__ __forceinline__ bool key_lt(const u64 (&a)[W], const u64 (&b)[W]) {   // unsigned multi-word a < b
    bool lt = false, eq = true;
#pragma unroll
    for (int q = 0; q < W; ++q) {
        lt = lt || (eq && a[q] < b[q]);
        eq = eq && a[q] == b[q];
    }
    return lt;
}

// One sweep over the sorted records, a small scan, and a kernel that copies the solid edges out, instead of one sweep
// whose tiles are chained by a decoupled look-back: a tile lives a few microseconds, and a chain that costs several
// L2 round trips per tile (measured: ~5 us of a ~9 us tile life) caps such a kernel far below the
// cost of the sweep itself.
//   sweep (this kernel)    : solid edges of every chunk -> chunk_sums[chunk]; statistics; into the stash (the sorter's
//                            spare buffer, 8 bytes per record at most) the place in the chunk and the multiplicity of
//                            every solid edge, in order
//   scan                   : chunk_sums -> exclusive prefix, total -> output cursor
//   count_write_kernel     : the solid edges copied out at out_base + prefix[chunk] + rank in chunk; only their keys
//                            are fetched again (1.34 -> 1.05 ms on config 2, where 3.6 % of the records end a solid
//                            run, against a second sweep that redid the arithmetic over all records)
//
// A chunk is kCountChunk consecutive records and belongs to ONE WARP, which walks it in rounds of 32 records, lane l
// holding record 32 r + l (coalesced loads, several rounds in flight). A record i is a run TAIL iff i == n-1 or
// key[i] != key[i+1] (the next key comes from the next lane by shuffle); the run ending at tail i has length
// i+1 - (start of the run), and the start is the place after the previous tail: the nearest lower tail of the round
// (one ballot, one find-leading-one) or the warp-uniform carry from the rounds before. For the run that is open at
// the chunk's first record the start is found by looking at the records right before it, 32 at a time, and, past
// 128 of them, by a 32-ary search for the first record equal to it (the records are sorted). So no state about runs
// travels between warps. Indices are chunk-relative u32 (modulo 2^32: if the range holds fewer than 2^32 records,
// run lengths come out right even when a run began long before the chunk).
constexpr u32 kCountChunk = 1024;        // records per warp
constexpr int kCountWarps = 8;           // warps per block
constexpr int kCountGroup = 4;           // rounds loaded ahead

template <int W>
__device__ __forceinline__ void shfl_key(u64 (&dst)[W], const u64 (&src)[W], int src_lane) {
#pragma unroll
    for (int q = 0; q < W; ++q) dst[q] = __shfl_sync(0xffffffffu, src[q], src_lane);
}

// WIDE: the range holds 2^32 records or more, so a run may be that long: run starts and lengths are 64-bit and the
// multiplicity saturates at 2^32-1 (reading A9); otherwise 32-bit modular arithmetic is exact.
template <int W, bool CSUM, bool WIDE>
__global__ void __launch_bounds__(kCountWarps * 32, W == 1 ? 6 : W == 2 ? 4 : 2) count_chunks_kernel(CountArgs a, DevState *st) {
    using len_t = std::conditional_t<WIDE, u64, u32>;
    constexpr int G = kCountGroup;
    __shared__ u64 s_red[3][kCountWarps];
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const u32 lt = lanemask_lt();
    const u64 chunk = (u64)blockIdx.x * kCountWarps + warp;
    const u64 c0 = chunk * kCountChunk;                     // global index of the chunk's first record
    u32 n_tails = 0, n_solid = 0;
    len_t sum_mult = 0;                                     // !WIDE: lengths of the runs ending in one chunk add up to < 2^32
    u64 csum = 0;
    if (c0 < a.n) {
        const u32 rem = (a.n - c0 < (u64)kCountChunk) ? (u32)(a.n - c0) : kCountChunk;   // records of this chunk
        const bool has_succ = c0 + kCountChunk < a.n;                                    // a record follows the chunk
        const u64 *kp = a.keys + c0 * W;
        auto load_round = [&](u32 r, u64 (&k)[W]) {         // record 32 r + lane, or zeros past the end of the data
            const u32 i = r * 32u + lane;
            if (i < rem || (i == rem && has_succ)) load_key<W>(kp, i, k);
            else {
#pragma unroll
                for (int q = 0; q < W; ++q) k[q] = 0;
            }
        };
        u64 key[G + 1][W];
        load_round(0, key[0]);

        // ---- start of the run that is open at the chunk's first record ----------------------------------------
        len_t carry = 0;                                     // chunk-relative start of the run in progress (modular)
        {
            u64 target[W], probe[W];
            shfl_key<W>(target, key[0], 0);
            // hi = lowest index known to belong to the run. Up to 4 rounds over the 32 records right below hi (these
            // lines were just read by the neighbouring warp), then a 32-ary search over all that lies below.
            u64 hi = c0;
            bool found = false;
#pragma unroll 1
            for (int r = 0; r < 4 && !found && hi > 0; ++r) {
                const bool inb = hi > (u64)lane;
                if (inb) load_key<W>(a.keys, hi - 1 - lane, probe);
                const u32 eqm = __ballot_sync(0xffffffffu, inb && !key_ne<W>(probe, target));
                const u32 lead = (eqm == 0xffffffffu) ? 32u : (u32)__ffs(~eqm) - 1u;   // equal records right below hi
                hi -= lead;
                found = lead < 32u;
            }
            if (!found && hi > 0) {
                u64 lo = 0;                                  // first index in [lo, hi] whose key is not less than target
                while (lo < hi) {
                    const u64 span = hi - lo;
                    const u64 p = span > 32 ? lo + (span / 33) * (lane + 1) : lo + lane;   // 32 probes, increasing with the lane
                    bool ge = true;
                    if (p < hi) { load_key<W>(a.keys, p, probe); ge = !key_lt<W>(probe, target); }
                    const u32 gem = __ballot_sync(0xffffffffu, ge);    // monotone: 0..0 1..1
                    const u32 f = gem ? (u32)__ffs(gem) - 1u : 32u;    // first probe inside the run (or none)
                    const u64 pf = __shfl_sync(0xffffffffu, p, (int)(f < 32u ? f : 31u));
                    const u64 pb = __shfl_sync(0xffffffffu, p, (int)(f ? f - 1u : 0u));
                    if (f < 32u && pf < hi) hi = pf;
                    if (f > 0u) lo = (pb < hi ? pb : hi - 1) + 1;      // the probe before the first hit is outside the run
                }
                hi = lo;
            }
            carry = (len_t)(hi - c0);                        // modular when the run began before the chunk
        }

        // ---- rounds --------------------------------------------------------------------------------------------
        // one round: FULL = every record of the round and its successor exist (no index checks)
        auto round = [&](auto full_tag, u32 r, const u64 (&k)[W], const u64 (&k_next_round)[W]) {
            constexpr bool FULL = decltype(full_tag)::value;
            const u32 i = r * 32u + lane;
            u64 kn[W];                                              // the record after mine: lane l+1, or lane 0 of the next round
#pragma unroll
            for (int q = 0; q < W; ++q) kn[q] = __shfl_sync(0xffffffffu, lane == 0 ? k_next_round[q] : k[q], (int)((lane + 1u) & 31u));
            bool tail = key_ne<W>(k, kn);
            if constexpr (!FULL) tail = i < rem && ((i + 1u == rem && !has_succ) || tail);
            const u32 T = __ballot_sync(0xffffffffu, tail);
            const u32 below = T & lt;
            const len_t start = below ? (len_t)(r * 32u + (32u - (u32)__clz(below))) : carry;   // place after the previous tail
            const len_t len = (len_t)(i + 1u) - start;
            bool solid = tail && len >= (len_t)a.d;
            const u32 S = __ballot_sync(0xffffffffu, solid);
            if (T) carry = (len_t)(r * 32u + (32u - (u32)__clz(T)));
            n_tails += (u32)__popc(T);
            if (solid)    // where the solid edge sits in its chunk and its multiplicity (A9: saturated), in chunk order
                a.stash[c0 + n_solid + (u32)__popc(S & lt)] = ((u64)i << 32) | (u64)((WIDE && len > (len_t)0xffffffffu) ? 0xffffffffu : (u32)len);
            n_solid += (u32)__popc(S);
            if (solid) sum_mult += len;
            if constexpr (CSUM) { if (tail) csum += (u64)len * mix_key<W>(k); }
        };
        if (rem == kCountChunk && c0 + kCountChunk + 32u <= a.n) {
            // full chunk with at least 32 records behind it: plain loads, G rounds in flight
#pragma unroll 1
            for (u32 r0 = 0; r0 < kCountChunk / 32u; r0 += G) {
#pragma unroll
                for (int g = 1; g <= G; ++g) load_key<W>(kp, (r0 + g) * 32u + lane, key[g]);
#pragma unroll
                for (int g = 0; g < G; ++g) round(std::true_type{}, r0 + g, key[g], key[g + 1]);
#pragma unroll
                for (int q = 0; q < W; ++q) key[0][q] = key[G][q];
            }
        } else {
            const u32 nrounds = (rem + 31u) / 32u;
#pragma unroll 1
            for (u32 r = 0; r < nrounds; ++r) {
                load_round(r + 1, key[1]);
                round(std::false_type{}, r, key[0], key[1]);
#pragma unroll
                for (int q = 0; q < W; ++q) key[0][q] = key[1][q];
            }
        }
    }
    {
        // per-warp and per-block numbers of solid edges; statistics: block reduction, one atomic per block and
        // counter, spread over 32 slots
        __shared__ u32 s_solid[kCountWarps];
        if constexpr (WIDE) sum_mult = (len_t)warp_reduce_add64((u64)sum_mult);
        else sum_mult = (len_t)__reduce_add_sync(0xffffffffu, (u32)sum_mult);
        if constexpr (CSUM) csum = warp_reduce_add64(csum);
        if (lane == 0) {
            s_red[0][warp] = n_tails; s_red[1][warp] = sum_mult; s_red[2][warp] = csum; s_solid[warp] = n_solid;
            reinterpret_cast<u32 *>(a.tile_sums + gridDim.x)[chunk] = n_solid;
        }
        __syncthreads();
        if (tid < 3) {
            u64 v = 0;
#pragma unroll
            for (int w = 0; w < kCountWarps; ++w) v += s_red[tid][w];
            if (v) atomicAdd(&a.stat_slots[(blockIdx.x & (kStatSlots - 1)) * kStatSlotWords + tid], v);
        } else if (tid == 32) {
            u64 v = 0;
#pragma unroll
            for (int w = 0; w < kCountWarps; ++w) v += s_solid[w];
            a.tile_sums[blockIdx.x] = v;
        }
    }
}

// tile_sums (one word per block of the sweeps = 64 KiB of records) -> exclusive prefix, in place; total added to the
// output cursor of the next range. One block, 4 words per thread and round.
__global__ void __launch_bounds__(1024) scan_tiles_kernel(u64 *tile_sums, u32 ntiles, DevState *st, int range_parity) {
    constexpr u32 PER = 4, ROUND = 1024 * PER;   // 32 contiguous bytes per thread: whole sectors
    __shared__ u64 s_w[32];
    __shared__ u64 s_carry;
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (u32 base = 0; base < ntiles; base += ROUND) {
        const u32 i0 = base + tid * PER;
        u64 v[PER], sum = 0;
#pragma unroll
        for (u32 j = 0; j < PER; ++j) { v[j] = (i0 + j < ntiles) ? tile_sums[i0 + j] : 0ull; sum += v[j]; }
        u64 incl = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u64 t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= (u32)o) incl += t;
        }
        if (lane == 31) s_w[warp] = incl;
        __syncthreads();
        u64 run = s_carry + incl - sum;
        for (u32 w = 0; w < warp; ++w) run += s_w[w];
#pragma unroll
        for (u32 j = 0; j < PER; ++j) { if (i0 + j < ntiles) tile_sums[i0 + j] = run; run += v[j]; }
        __syncthreads();
        if (tid == 1023) s_carry = run;
        __syncthreads();
    }
    if (tid == 0) {
        if (range_parity < 0) st->merge_heads = s_carry;   // sdbg_build's merge: number of distinct keys
        else st->out_cursor[range_parity ^ 1] = st->out_cursor[range_parity] + s_carry;
    }
}

// Sweep 2 when sweep 1 has left a stash (the spare buffer of the sorter: one 8-byte entry per record at most, chunk by
// chunk): the solid edges of a chunk are copied out from their (place in chunk, multiplicity) entries — the sorted
// records are not read a second time, only the keys of the solid edges are fetched (they are a few per cent of the
// records and their lines were read microseconds ago).
template <int W>
__global__ void __launch_bounds__(kCountWarps * 32) count_write_kernel(CountArgs a, const DevState *st) {
    const u32 lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const u64 chunk = (u64)blockIdx.x * kCountWarps + warp;
    const u64 c0 = chunk * kCountChunk;
    if (c0 >= a.n) return;
    const u32 *ws = reinterpret_cast<const u32 *>(a.tile_sums + gridDim.x) + (u64)blockIdx.x * kCountWarps;
    u64 out_pos = st->out_cursor[a.range_parity] + a.tile_sums[blockIdx.x];
    for (u32 w = 0; w < warp; ++w) out_pos += ws[w];
    const u32 cnt = ws[warp];
    for (u32 e = lane; e < cnt; e += 32u) {
        const u64 ent = a.stash[c0 + e];
        const u64 pos = out_pos + e;
        if (pos < a.out_cap) {
            u64 k[W];
            load_key<W>(a.keys, c0 + (ent >> 32), k);
#pragma unroll
            for (int q = 0; q < W; ++q) a.out_keys[pos * W + q] = k[q];
            a.out_mult[pos] = (u32)ent;
        }
    }
}

u64 count_tile_records(u32) { return kCountChunk; }

template <int W>
static int launch_count_w(const CountArgs &a, DevState *st, cudaStream_t s) {
    const u64 chunks = (a.n + kCountChunk - 1) / kCountChunk;
    if (chunks == 0) return 0;
    const u64 blocks = (chunks + kCountWarps - 1) / kCountWarps;
    if (blocks > 0x7fffffffull) return (int)cudaErrorInvalidValue;
    const bool wide = a.n > 0xffffffffull || a.force_wide;
    const unsigned g = (unsigned)blocks, t = kCountWarps * 32;
    if (wide) {
        if (a.want_csum) count_chunks_kernel<W, true, true><<<g, t, 0, s>>>(a, st);
        else             count_chunks_kernel<W, false, true><<<g, t, 0, s>>>(a, st);
    } else {
        if (a.want_csum) count_chunks_kernel<W, true, false><<<g, t, 0, s>>>(a, st);
        else             count_chunks_kernel<W, false, false><<<g, t, 0, s>>>(a, st);
    }
    scan_tiles_kernel<<<1, 1024, 0, s>>>(a.tile_sums, (u32)blocks, st, a.range_parity);
    count_write_kernel<W><<<g, t, 0, s>>>(a, st);
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
// Same shape as the count sweeps: one warp per 1,024-record chunk, rounds of 32 records.
//   sweep 1 (WRITE = false): heads (records that differ from their predecessor) per chunk and per block
//   scan                   : block sums -> exclusive prefix; total -> st->merge_heads
//   sweep 2 (WRITE = true) : distinct index of a record = heads before it (inclusive) - 1; heads write their key; the
//                            multiplicities of a run are added up inside the round by a segmented scan over the lanes,
//                            and the last lane of a segment writes its sum into acc[distinct index]: with a plain store
//                            when the whole run lies inside the round, with an atomic add when the run crosses a round.
//   finish                 : acc (u64, zeroed before) saturates into out_mult (u32, reading A9).
template <int W, bool WRITE>
__global__ void __launch_bounds__(kCountWarps * 32) merge_chunks_kernel(MergeArgs a, DevState *st) {
    __shared__ u32 s_heads[kCountWarps];
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const u32 le = lanemask_lt() | (1u << lane);
    const u64 chunk = (u64)blockIdx.x * kCountWarps + warp;
    const u64 c0 = chunk * kCountChunk;
    u32 n_heads = 0;
    u64 *block_sums = a.sums;
    u32 *chunk_sums = reinterpret_cast<u32 *>(a.sums + gridDim.x);
    if (c0 < a.n) {
        const u32 rem = (a.n - c0 < (u64)kCountChunk) ? (u32)(a.n - c0) : kCountChunk;
        u64 base = 0;                                        // heads before this chunk
        if constexpr (WRITE) {
            base = block_sums[blockIdx.x];
            for (u32 w = 0; w < warp; ++w) base += chunk_sums[(u64)blockIdx.x * kCountWarps + w];
        }
        u64 carry_key[W];                                    // the record before the round's first one (lane 0 uses it)
        const bool first_chunk = c0 == 0;
        if (!first_chunk) load_key<W>(a.keys, c0 - 1, carry_key);
        else {
#pragma unroll
            for (int q = 0; q < W; ++q) carry_key[q] = 0;
        }
        const u32 nrounds = (rem + 31u) / 32u;
#pragma unroll 1
        for (u32 r = 0; r < nrounds; ++r) {
            const u32 i = r * 32u + lane;
            const bool valid = i < rem;
            u64 k[W], kp[W];
            if (valid) load_key<W>(a.keys, c0 + i, k);
            else {
#pragma unroll
                for (int q = 0; q < W; ++q) k[q] = 0;
            }
#pragma unroll
            for (int q = 0; q < W; ++q) {
                const u64 up = __shfl_up_sync(0xffffffffu, k[q], 1);
                kp[q] = lane == 0 ? carry_key[q] : up;
            }
            const bool head = valid && ((first_chunk && i == 0) || key_ne<W>(k, kp));
            const u32 H = __ballot_sync(0xffffffffu, head);
            if constexpr (!WRITE) {
                n_heads += (u32)__popc(H);
            } else {
                const u32 V = __ballot_sync(0xffffffffu, valid);
                const u64 di = base + n_heads + (u32)__popc(H & le) - 1u;   // n_heads: heads of the earlier rounds
                if (head) {
#pragma unroll
                    for (int q = 0; q < W; ++q) a.out_keys[di * W + q] = k[q];
                }
                // inclusive sum of mult over the lanes of my segment (segments begin at heads and at lane 0)
                u64 s = valid ? (u64)a.mult[c0 + i] : 0ull;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const u64 t = __shfl_up_sync(0xffffffffu, s, o);
                    const u32 between = le & ~(le >> o);                  // lanes (lane-o, lane]
                    if (lane >= (u32)o && (H & between) == 0) s += t;     // no head in between: same segment
                }
                // last lane of a segment: the next lane is a head, or there is no next valid lane in the round
                const bool seg_last = valid && (lane == 31u || ((H >> (lane + 1u)) & 1u) || !((V >> (lane + 1u)) & 1u));
                if (seg_last) {
                    const bool whole = (H & le) != 0 && lane != 31u && ((H >> (lane + 1u)) & 1u);   // began and ended inside the round
                    if (whole) a.acc[di] = s;
                    else atomicAdd(&a.acc[di], s);
                }
                n_heads += (u32)__popc(H);
            }
            const u32 last = 31u;                            // the round's last record (only read by a following round: full)
#pragma unroll
            for (int q = 0; q < W; ++q) carry_key[q] = __shfl_sync(0xffffffffu, k[q], (int)last);
        }
    }
    if constexpr (!WRITE) {
        if (lane == 0) {
            s_heads[warp] = n_heads;
            chunk_sums[chunk] = n_heads;
        }
        __syncthreads();
        if (tid == 0) {
            u64 v = 0;
#pragma unroll
            for (int w = 0; w < kCountWarps; ++w) v += s_heads[w];
            block_sums[blockIdx.x] = v;
        }
    }
}

__global__ void __launch_bounds__(256) merge_finish_kernel(const u64 *acc, u32 *out_mult, u64 n, const DevState *st) {
    const u64 m = st->merge_heads;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < m && i < n; i += (u64)gridDim.x * blockDim.x)
        out_mult[i] = acc[i] > 0xffffffffull ? 0xffffffffu : (u32)acc[i];
}

u64 merge_tile_records() { return kCountChunk; }

template <int W>
static void launch_merge_w(const MergeArgs &a, DevState *st, cudaStream_t s) {
    const u64 chunks = (a.n + kCountChunk - 1) / kCountChunk, blocks = (chunks + kCountWarps - 1) / kCountWarps;
    merge_chunks_kernel<W, false><<<(unsigned)blocks, kCountWarps * 32, 0, s>>>(a, st);
    scan_tiles_kernel<<<1, 1024, 0, s>>>(a.sums, (u32)blocks, st, -1);
    merge_chunks_kernel<W, true><<<(unsigned)blocks, kCountWarps * 32, 0, s>>>(a, st);
}

void launch_merge(const MergeArgs &a, DevState *st, cudaStream_t s) {
    if (a.n == 0) return;
    switch (a.W) {
        case 1: launch_merge_w<1>(a, st, s); break;
        case 2: launch_merge_w<2>(a, st, s); break;
        case 3: launch_merge_w<3>(a, st, s); break;
        case 4: launch_merge_w<4>(a, st, s); break;
    }
    u64 blocks = (a.n + 255) / 256;
    if (blocks > (u64)num_sms() * 8) blocks = (u64)num_sms() * 8;
    merge_finish_kernel<<<(unsigned)blocks, 256, 0, s>>>(a.acc, a.out_mult, a.n, st);
}

}  // namespace sdbg

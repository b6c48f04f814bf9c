// hashcount.cu — step a4 for records that are sorted by their TOP key bytes only: "all (k+1)-mers
// from the input reads are sorted and counted ... only (k+1)-mers that appear at least d (2 by default) times are
// kept" (§2 ¶4). This is the paper's own partition idea (the k-mers are partitioned by a
// length-l prefix and consecutive partitions are handled together) carried one level down: after P_hi radix passes over
// the most significant key bytes all copies of an edge lie inside one run of equal top bytes (a bucket), and a segment
// of consecutive whole buckets is small enough to be counted in SHARED memory. One CTA per segment:
//   1 every record of the segment is inserted into an open-addressing table of (key, count) slots in shared memory;
//   2 the slots with count >= d are put in key order inside shared memory (one pass of order-preserving binning, then
//     insertion inside the tiny bins) — buckets are consecutive in key order and segments too, so the ordered solid edges
//     of a segment are a contiguous piece of the final output;
//   3 they are written, with their counts, to the place of the segment in a staging buffer, and the number of them to
//     seg_count[segment]; a scan and a copy kernel (hash_scan_kernel, hash_copy_kernel) append them in order.
// Nothing but the solid edges goes through any further pass. Segment borders are found by hash_bounds_kernel.
// Whatever does not fit (a bucket longer than the search window, a full table, more solid edges than sort places)
// raises *overflow; the caller then sorts the range the plain way (api_count.inc), so the result is the same.
#include "kernels.cuh"

namespace sdbg {

constexpr u64 kEmpty = ~0ull;   // an all-ones key (edge T...T at k = 31) is counted beside the table

// first index i in [lo, hi] with (keys[i] >> shift) != t, where the predicate is monotone on [lo, hi) and taken as
// true at hi; one warp, 32-ary search (every lane returns the result)
__device__ __forceinline__ u64 warp_first_other(const u64 *__restrict__ keys, u64 lo, u64 hi, u32 shift, u64 t) {
    const u32 lane = lane_id();
    while (hi - lo >= 32) {
        const u64 stride = (hi - lo + 31) / 32;
        u64 p = lo + (u64)(lane + 1) * stride - 1;      // probes lo+stride-1, lo+2*stride-1, ..., clamped to hi-1
        if (p > hi - 1) p = hi - 1;
        const u32 b = __ballot_sync(0xffffffffu, (keys[p] >> shift) != t);
        if (b == 0) { lo = hi; break; }                  // no record of [lo, hi) differs
        const u32 f = __ffs(b) - 1;                      // the answer lies behind probe f-1 and not behind probe f
        hi = __shfl_sync(0xffffffffu, p, f);
        lo = lo + (u64)f * stride;
    }
    const u64 p = lo + lane;
    const u32 b = __ballot_sync(0xffffffffu, p < hi ? (keys[p] >> shift) != t : true);   // lane hi-lo <= 31 says true
    return lo + (u64)(__ffs(b) - 1);
}

// seg_start[c], c in [0, nchunks]: the first bucket border at or after record c * chunk (n for c = nchunks). A bucket
// that runs on for more than `window` records past the nominal place raises *overflow.
__global__ void __launch_bounds__(256) hash_bounds_kernel(const u64 *__restrict__ keys, u64 n, u32 shift, u32 chunk, u32 window,
                                                          u64 nchunks, u64 *__restrict__ seg_start, u32 *overflow) {
    const u64 c = (u64)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (c > nchunks) return;
    u64 res;
    const u64 x = c * chunk;
    if (c == 0) res = 0;
    else if (x >= n) res = n;
    else {
        const u64 t = keys[x - 1] >> shift;
        if ((keys[x] >> shift) != t) res = x;
        else {
            const u64 lim = x + window < n ? x + window : n;
            res = warp_first_other(keys, x, lim, shift, t);
            if (res == lim && lim < n && lane_id() == 0) atomicOr(overflow, 1u);   // not a border (or unknown): give up
        }
    }
    if (lane_id() == 0) seg_start[c] = res;
}

// U = loads in flight per thread; PACK16: counts are 16-bit halves of u32 words (a segment has at most window + chunk
// < 65,536 records), which brings the short-bucket shape to 52 KiB and four CTAs per SM
template <int THREADS, int MINB, int U, bool PACK16>
__global__ void __launch_bounds__(THREADS, MINB)
hash_count_kernel(HashCountArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    u64 *t_key = reinterpret_cast<u64 *>(smem_raw);                  // u64[table_slots]
    u32 *t_cnt = reinterpret_cast<u32 *>(smem_raw + (size_t)a.table_slots * 8); // u32[table_slots] (PACK16: u16 pairs)
    constexpr u32 CB = PACK16 ? 2u : 4u;                              // bytes of a count
    __shared__ u32 s_ones, s_full, s_nsolid, s_distinct;
    __shared__ u64 s_sum;
    const u32 tid = threadIdx.x;
    const u64 seg = blockIdx.x;
    const u64 s = a.seg_start[seg], e = a.seg_start[seg + 1];
    if (e <= s) { if (tid == 0) a.seg_count[seg] = 0; return; }
    const u64 kfirst = a.keys[s] >> a.top_shift, klast = a.keys[e - 1] >> a.top_shift;   // first and last bucket of the segment
    // the first U records of every thread are on their way while the table is cleared
    u64 kq[U];
#pragma unroll
    for (int u = 0; u < U; ++u) { const u64 i = s + (u64)u * THREADS + tid; kq[u] = i < e ? ld_stream(a.keys + i) : 0ull; }
    // table size: the power of two from 1.5 x the records of the segment on (all of them might be distinct)
    u32 TS = 1024;
    while (TS < a.table_slots && (u64)TS * 2 < (e - s) * 3) TS <<= 1;
    const u32 mask = TS - 1u, hshift = 32u - (u32)__ffs(TS) + 1u;
    {
        uint4 *k4 = reinterpret_cast<uint4 *>(t_key), *c4 = reinterpret_cast<uint4 *>(t_cnt);
        const uint4 ones = make_uint4(~0u, ~0u, ~0u, ~0u), zero = make_uint4(0u, 0u, 0u, 0u);
        for (u32 i = tid; i < TS / 2; i += THREADS) k4[i] = ones;
        for (u32 i = tid; i < TS * CB / 16; i += THREADS) c4[i] = zero;
    }
    if (tid == 0) { s_ones = 0; s_full = 0; s_nsolid = 0; s_distinct = 0; s_sum = 0; }
    __syncthreads();

    // ---- 1: insert ---------------------------------------------------------------------------------------------------
    u32 created = 0;
    const bool may_ones = klast == (~0ull >> a.top_shift);            // only the last bucket of all can hold the all-ones key
    auto insert = [&](u64 key) {
        if (may_ones && key == kEmpty) { atomicAdd(&s_ones, 1u); return; }
        u32 h = ((u32)key ^ (u32)(key >> 32)) * 0x9E3779B1u;
        h ^= (u32)(key >> 20);
        u32 slot = (h * 0x85EBCA6Bu) >> hshift;
        for (u32 probes = 0;; ++probes) {
            u64 cur = t_key[slot];
            if (cur == kEmpty) {
                cur = atomicCAS(&t_key[slot], kEmpty, key);
                if (cur == kEmpty) { ++created; cur = key; }
            }
            if (cur == key) {
                if constexpr (PACK16) atomicAdd(&t_cnt[slot >> 1], 1u << ((slot & 1u) * 16u));
                else atomicAdd(&t_cnt[slot], 1u);
                break;
            }
            slot = (slot + 1u) & mask;
            if (probes >= TS) { s_full = 1; break; }
        }
    };
    // a segment has fewer than 2^16 records: 32-bit positions relative to its start
    const u32 m = (u32)(e - s);
    for (u32 base = 0;;) {
        const u32 rem = m - base > tid ? m - base - tid : 0u;          // my records of this round: u * THREADS < rem
#pragma unroll
        for (int u = 0; u < U; ++u) if ((u32)u * THREADS < rem) insert(kq[u]);
        base += (u32)U * THREADS;
        if (base >= m) break;
        const u64 *src = a.keys + s + base + tid;
        const u32 rem2 = m - base > tid ? m - base - tid : 0u;
#pragma unroll
        for (int u = 0; u < U; ++u) kq[u] = (u32)u * THREADS < rem2 ? ld_stream(src + u * THREADS) : 0ull;
    }
    if (created) atomicAdd(&s_distinct, created);
    __syncthreads();
    if (s_full) { if (tid == 0) { atomicOr(a.overflow, 2u); a.seg_count[seg] = 0; } return; }

    // ---- 2: the solid slots, compacted to the front of a list in shared memory (reusing the table in place is not
    //         possible while it is read, so the list lives behind it) ------------------------------------------------------
    u64 *l_key = reinterpret_cast<u64 *>(smem_raw + (size_t)a.table_slots * (8 + CB));    // u64[max_solid]
    u32 *l_cnt = reinterpret_cast<u32 *>(smem_raw + (size_t)a.table_slots * (8 + CB) + (size_t)a.max_solid * 8);
    u64 sum = 0;
    {   // the live part of the table, 16 bytes of counts (4 or 8 slots) per load; most vectors hold no solid edge
        constexpr u32 SPV = PACK16 ? 8u : 4u;
        const uint4 *c4 = reinterpret_cast<const uint4 *>(t_cnt);
        const u32 d = a.d;
        for (u32 v = tid; v < TS / SPV; v += THREADS) {
            const uint4 w = c4[v];
            u32 cs[SPV];
            if constexpr (PACK16) {
                cs[0] = w.x & 0xffffu; cs[1] = w.x >> 16; cs[2] = w.y & 0xffffu; cs[3] = w.y >> 16;
                cs[4] = w.z & 0xffffu; cs[5] = w.z >> 16; cs[6] = w.w & 0xffffu; cs[7] = w.w >> 16;
            } else {
                cs[0] = w.x; cs[1] = w.y; cs[2] = w.z; cs[3] = w.w;
            }
            u32 mx = 0;
#pragma unroll
            for (u32 q = 0; q < SPV; ++q) mx = cs[q] > mx ? cs[q] : mx;
            if (mx < d) continue;
#pragma unroll
            for (u32 q = 0; q < SPV; ++q) {
                if (cs[q] >= d) {
                    const u32 p = atomicAdd(&s_nsolid, 1u);
                    if (p < a.max_solid) { l_key[p] = t_key[v * SPV + q]; l_cnt[p] = cs[q]; }
                    sum += cs[q];
                }
            }
        }
    }
    if (tid == 0 && s_ones) {
        ++s_distinct;                                    // nobody else touches it between the barriers
        if (s_ones >= a.d) {
            const u32 p = atomicAdd(&s_nsolid, 1u);
            if (p < a.max_solid) { l_key[p] = kEmpty; l_cnt[p] = s_ones; }
            sum += s_ones;
        }
    }
    sum = warp_reduce_add64(sum);
    if ((tid & 31u) == 0 && sum) atomicAdd(&s_sum, sum);
    __syncthreads();
    const u32 ns = s_nsolid;
    if (ns > a.max_solid) { if (tid == 0) { atomicOr(a.overflow, 4u); a.seg_count[seg] = 0; } return; }
    if (tid == 0) {
        a.seg_count[seg] = ns;
        u64 *slot = a.stat_slots + (size_t)(blockIdx.x & (kStatSlots - 1)) * kStatSlotWords;
        atomicAdd(&slot[0], (u64)s_distinct);
        if (s_sum) atomicAdd(&slot[1], s_sum);
    }
    if (ns == 0) return;

    // ---- 3: order the list by key. The solid edges of a segment are spread evenly over its key range, so one pass of
    //         order-preserving binning (1,024 bins over the range of the segment's buckets) leaves bins of one or two
    //         entries, which the owner of the bin puts in order by insertion. The table is dead: bins and the ordered
    //         list live in its place. -----------------------------------------------------------------------------------
    constexpr int NB = 1024, Q = NB / THREADS;                        // bins (also the most entries of a segment); per thread
    u32 *bins = t_cnt;
    u64 *o_key = t_key;
    u32 *o_cnt = reinterpret_cast<u32 *>(t_key + NB);
    const u64 k0 = kfirst << a.top_shift;
    const u64 rm1 = ((klast - kfirst + 1ull) << a.top_shift) - 1ull;  // largest offset inside the segment's buckets
    const int sh0 = 54 - __clzll((long long)rm1), sh = sh0 > 0 ? sh0 : 0;   // (rm1 >> sh) < 1024
#pragma unroll
    for (int q = 0; q < Q; ++q) bins[tid + q * THREADS] = 0;
    __syncthreads();
    u32 myb[Q], myr[Q];
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        const u32 i = tid + q * THREADS;
        myb[q] = 0; myr[q] = 0;
        if (i < ns) { myb[q] = (u32)((l_key[i] - k0) >> sh); myr[q] = atomicAdd(&bins[myb[q]], 1u); }
    }
    __syncthreads();
    __shared__ u32 s_w[THREADS / 32];
    u32 c[Q], csum = 0;
#pragma unroll
    for (int q = 0; q < Q; ++q) { c[q] = bins[Q * tid + q]; csum += c[q]; }
    const u32 incl = warp_incl_scan_add(csum);
    if ((tid & 31u) == 31u) s_w[tid >> 5] = incl;
    __syncthreads();
    u32 base0 = incl - csum;
    for (u32 w = 0; w < (tid >> 5); ++w) base0 += s_w[w];
    {
        u32 run = base0;
#pragma unroll
        for (int q = 0; q < Q; ++q) { bins[Q * tid + q] = run; run += c[q]; }
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        const u32 i = tid + q * THREADS;
        if (i < ns) { const u32 p = bins[myb[q]] + myr[q]; o_key[p] = l_key[i]; o_cnt[p] = l_cnt[i]; }
    }
    __syncthreads();
    {
        u32 b0 = base0;
#pragma unroll
        for (int q = 0; q < Q; ++q) {
            for (u32 x = 1; x < c[q]; ++x) {                           // insertion sort of places [b0, b0 + c)
                const u64 kx = o_key[b0 + x]; const u32 cx = o_cnt[b0 + x];
                u32 y = x;
                while (y > 0 && o_key[b0 + y - 1] > kx) { o_key[b0 + y] = o_key[b0 + y - 1]; o_cnt[b0 + y] = o_cnt[b0 + y - 1]; --y; }
                o_key[b0 + y] = kx; o_cnt[b0 + y] = cx;
            }
            b0 += c[q];
        }
    }
    __syncthreads();
    // ---- write the sorted solid edges of the segment to its place in the staging buffer ---------------------------------
    // staging (8 bytes per record, the sorter's spare buffer): the segment owns places [s, e); its ns <= (e - s) / d solid
    // keys (d >= 2) fill the first half at most, their u32 counts start at the middle place
    u32 *stage_cnt = reinterpret_cast<u32 *>(a.stage_keys + s + ((e - s + 1) >> 1));
    for (u32 i = tid; i < ns; i += THREADS) { a.stage_keys[s + i] = o_key[i]; stage_cnt[i] = o_cnt[i]; }
}

// seg_count -> exclusive prefix in place (u64), total to *total; one block, tiles of 4,096 (the array has n / chunk
// entries: 97 k on config 2, 1.5 M on config 3)
__global__ void __launch_bounds__(1024) hash_scan_kernel(u64 *__restrict__ seg_count, u64 nseg, u64 *total) {
    __shared__ u64 s_w[32];
    __shared__ u64 s_carry;
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (u64 base = 0; base < nseg; base += 4096) {
        const u64 i = base + 4ull * tid;
        u64 v[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) v[q] = i + q < nseg ? seg_count[i + q] : 0;
        const u64 sum = v[0] + v[1] + v[2] + v[3];
        u64 incl = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            u64 t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= (u32)o) incl += t;
        }
        if (lane == 31) s_w[warp] = incl;
        __syncthreads();
        u64 off = s_carry;
        for (u32 w = 0; w < warp; ++w) off += s_w[w];
        u64 run = off + incl - sum;
#pragma unroll
        for (int q = 0; q < 4; ++q) { if (i + q < nseg) seg_count[i + q] = run; run += v[q]; }
        __syncthreads();
        if (tid == 1023) s_carry = off + incl;
        __syncthreads();
    }
    if (tid == 0) *total = s_carry;
}

// the staged solid edges of every segment appended to the output, in segment (= key) order; one warp per segment
__global__ void __launch_bounds__(256) hash_copy_kernel(HashCountArgs a, const u64 *__restrict__ total, DevState *st, int range_parity) {
    const u64 base = st->out_cursor[range_parity];
    const u32 lane = lane_id();
    for (u64 seg = (u64)blockIdx.x * 8 + (threadIdx.x >> 5); seg < a.nseg; seg += (u64)gridDim.x * 8) {
        const u64 off = a.seg_count[seg];
        const u64 cnt = (seg + 1 < a.nseg ? a.seg_count[seg + 1] : *total) - off;
        const u64 s = a.seg_start[seg], e = a.seg_start[seg + 1];
        const u32 *stage_cnt = reinterpret_cast<const u32 *>(a.stage_keys + s + ((e - s + 1) >> 1));
        for (u64 i = lane; i < cnt; i += 32) {
            const u64 pos = base + off + i;
            if (pos < a.out_cap) { a.out_keys[pos] = a.stage_keys[s + i]; a.out_mult[pos] = stage_cnt[i]; }
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) st->out_cursor[range_parity ^ 1] = base + *total;
}

// two shapes: big segments (chunk 4,096: one or two long buckets) 512 threads x 2 CTAs per SM with 8,192 slots; small
// segments (chunk 2,048: many short buckets) 256 threads x 4 CTAs per SM with 4,096 slots and 16-bit counts
u64 hash_smem_bytes(u32 table_slots, u32 max_solid) { return (u64)table_slots * (table_slots > 4096 ? 12 : 10) + (u64)max_solid * 12; }

int hash_setup() {
    int e = (int)cudaFuncSetAttribute(hash_count_kernel<512, 2, 8, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 110 * 1024);
    if (e) return e;
    return (int)cudaFuncSetAttribute(hash_count_kernel<256, 4, 9, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 54 * 1024);
}

void launch_hash_bounds(const HashCountArgs &a, cudaStream_t s) {
    const u64 warps = a.nseg + 1, blocks = (warps + 7) / 8;
    hash_bounds_kernel<<<(unsigned)blocks, 256, 0, s>>>(a.keys, a.n, a.top_shift, a.chunk, a.window, a.nseg, a.seg_start, a.overflow);
}
int launch_hash_count(const HashCountArgs &a, cudaStream_t s) {
    if (a.nseg == 0 || a.nseg > 0x7fffffffull || a.max_solid != 1024 || (u64)a.window + a.chunk >= 65536) return (int)cudaErrorInvalidValue;
    const size_t smem = hash_smem_bytes(a.table_slots, a.max_solid);
    if (a.table_slots > 4096) hash_count_kernel<512, 2, 8, false><<<(unsigned)a.nseg, 512, smem, s>>>(a);
    else hash_count_kernel<256, 4, 9, true><<<(unsigned)a.nseg, 256, smem, s>>>(a);
    return (int)cudaGetLastError();
}
void launch_hash_append(const HashCountArgs &a, u64 *total, DevState *st, int range_parity, cudaStream_t s) {
    hash_scan_kernel<<<1, 1024, 0, s>>>(a.seg_count, a.nseg, total);
    const u64 blocks = (a.nseg + 7) / 8;
    hash_copy_kernel<<<(unsigned)blocks, 256, 0, s>>>(a, total, st, range_parity);
}

}  // namespace sdbg

// hashcount.cu — step a4 for records that are sorted by their TOP key bytes only: "all (k+1)-mers
// from the input reads are sorted and counted ... only (k+1)-mers that appear at least d (2 by default) times are
// kept" (§2 ¶4). This is the paper's own partition idea (the k-mers are partitioned by a
// length-l prefix and consecutive partitions are handled together) carried one level down: after P_hi radix passes over
// the most significant key bytes all copies of an edge lie inside one run of equal top bytes (a bucket), and a segment
// of consecutive whole buckets is small enough to be counted in SHARED memory. Persistent CTAs take segments by atomic
// ticket (two ahead, so that neither the ticket nor the bounds of a segment are ever waited for); per segment:
//   1 every record of the segment is inserted into an open-addressing table of (key, 16-bit count) slots in shared memory.
//     A warp holds U rows of 32 records at a time and first tries the HOME slot of all of them (one ATOMS.CAS.64 that
//     installs the key or returns what is there, then one ATOMS.ADD on the count) with no loop and no divergence; the few
//     records whose home slot holds another key are then finished in ONE divergent probing loop per group of rows;
//   2 the slots with count >= d are put in key order inside shared memory (one pass of order-preserving binning, then
//     insertion inside the tiny bins) — buckets are consecutive in key order and segments too, so the ordered solid edges
//     of a segment are a contiguous piece of the final output;
//   3 they are written, with their counts, to the place of the segment in a staging buffer (the sorter's spare buffer),
//     the number of them to seg_count[segment] and added to the sum of its block of 64 segments. hash_scan_kernel (one
//     block: prefix of the block sums) and hash_copy_kernel (a CTA per block of segments: prefix inside the block, then a
//     warp per segment) append them in order. CTAs never wait for one another: a chain of solid counts through the
//     segments (decoupled look-back, tried first) made all resident segments resolve in lockstep, each walk some ten L2
//     round trips long, and cost a quarter of the kernel's time; staging costs 24 bytes per solid edge of HBM traffic.
// The first records of the NEXT segment are requested before step 2, so loads are in flight while a CTA sorts.
// Nothing but the solid edges goes through any further pass. Segment borders are found by hash_bounds_kernel.
// Whatever does not fit (a bucket longer than the search window, a full table, more solid edges than sort places, two keys
// of several words with one stand-in) raises *overflow; the caller then sorts the range the plain way (api_count.inc), so
// the result is the same. Keys of several words: see "keys of W > 1 words" below.
#include "kernels.cuh"
#include <type_traits>

namespace sdbg {

constexpr u64 kEmpty = ~0ull;   // an all-ones key (edge T...T at k = 31) is counted beside the table

// first record i in [lo, hi] (records of W words, the first one compared) with (keys[i W] >> shift) != t, where the predicate is monotone on [lo, hi) and taken as
// true at hi; one warp, 32-ary search (every lane returns the result)
__device__ __forceinline__ u64 warp_first_other(const u64 *__restrict__ keys, u32 W, u64 lo, u64 hi, u32 shift, u64 t) {
    const u32 lane = lane_id();
    while (hi - lo >= 32) {
        const u64 stride = (hi - lo + 31) / 32;
        u64 p = lo + (u64)(lane + 1) * stride - 1;      // probes lo+stride-1, lo+2*stride-1, ..., clamped to hi-1
        if (p > hi - 1) p = hi - 1;
        const u32 b = __ballot_sync(0xffffffffu, (keys[p * W] >> shift) != t);
        if (b == 0) { lo = hi; break; }                  // no record of [lo, hi) differs
        const u32 f = __ffs(b) - 1;                      // the answer lies behind probe f-1 and not behind probe f
        hi = __shfl_sync(0xffffffffu, p, f);
        lo = lo + (u64)f * stride;
    }
    const u64 p = lo + lane;
    const u32 b = __ballot_sync(0xffffffffu, p < hi ? (keys[p * W] >> shift) != t : true);   // lane hi-lo <= 31 says true
    return lo + (u64)(__ffs(b) - 1);
}

// seg_start[c], c in [0, nchunks]: the first bucket border at or after record c * chunk (n for c = nchunks). A bucket
// that runs on for more than `window` records past the nominal place raises *overflow.
__global__ void __launch_bounds__(256) hash_bounds_kernel(const u64 *__restrict__ keys, u32 W, u64 n, u32 shift, u32 chunk, u32 window,
                                                          u64 nchunks, u64 *__restrict__ seg_start, u32 *overflow) {
    const u64 c = (u64)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (c > nchunks) return;
    u64 res;
    const u64 x = c * chunk;
    if (c == 0) res = 0;
    else if (x >= n) res = n;
    else {
        const u64 t = keys[(x - 1) * W] >> shift;
        if ((keys[x * W] >> shift) != t) res = x;
        else {
            const u64 lim = x + window < n ? x + window : n;
            res = warp_first_other(keys, W, x, lim, shift, t);
            if (res == lim && lim < n && lane_id() == 0) atomicOr(overflow, 1u);   // not a border (or unknown): give up
        }
    }
    if (lane_id() == 0) seg_start[c] = res;
}

constexpr u32 kSegBlock = kHashSegBlock;   // segments per block sum (hash_scan_kernel, hash_copy_kernel)

__device__ __forceinline__ u32 hash_slot(u64 key, u32 hshift) {
    const u32 h = (u32)key + (u32)(key >> 32) * 0x9E3779B1u;
    return (h * 0x85EBCA6Bu) >> hshift;
}

// shared-memory accesses by 32-bit shared address (no generic-to-shared conversion per access)
__device__ __forceinline__ u64 s_cas64(u32 addr, u64 cmp, u64 val) {
    u64 r;
    asm volatile("atom.shared.cas.b64 %0, [%1], %2, %3;" : "=l"(r) : "r"(addr), "l"(cmp), "l"(val) : "memory");
    return r;
}
template <int OFS>
__device__ __forceinline__ void s_red_add(u32 addr, u32 v) {
    asm volatile("red.shared.add.u32 [%0+%2], %1;" ::"r"(addr), "r"(v), "n"(OFS) : "memory");
}

// ---- keys of W > 1 words ------------------------------------------------------------------------------------------------------
// The records stay where the extractor wrote them (a.recs, any order). What is sorted by the top passes and counted here
// is a one-word STAND-IN of every record (a.keys: the top bits of its first word, which the passes look at, and below
// them a fingerprint of the whole key; common.cuh pair_key) with the index of the record as payload (a.vals): 12 bytes
// move per record and pass instead of 8 W. The table holds stand-ins, and beside each the place (in the segment) of the
// record that installed it. Equal keys have equal stand-ins; that equal stand-ins are equal keys is CHECKED for every
// record that did not install its slot (word by word against the record that did: two reads through the indices), and a
// mismatch raises *overflow like everything else that does not fit, so the result stays exact. Records that are alone in
// their slot (most of them at large k) are never read here at all.
// Keys of TWO words are their own stand-ins: whole records (16 bytes against the 12 of a pair) go through the top passes, a.keys
// holds them, sorted, a.vals is null, the fingerprint is made here when a record is loaded, and the check reads the record
// that installed the slot a few hundred bytes away instead of somewhere in HBM — on reads where half of the records are
// copies the random reads of the pair path cost more than the 4 extra bytes per pass.
// 16 bytes of a record read at a random place: the L2 is told to fetch 64 bytes around it, not the 128 of its default
__device__ __forceinline__ ulonglong2 ld_rec16(const u64 *p) {
    ulonglong2 v;
    asm volatile("ld.global.L2::64B.v2.u64 {%0,%1}, [%2];" : "=l"(v.x), "=l"(v.y) : "l"(p));
    return v;
}
template <int W>
__device__ __forceinline__ void load_key(const u64 *__restrict__ src, u64 (&k)[W]) {   // src = first word of the record
    if constexpr (W == 1) k[0] = ld_stream(src);
    else if constexpr (W == 2) { const ulonglong2 v = ld_rec16(src); k[0] = v.x; k[1] = v.y; }
    else if constexpr (W == 4) {
        const ulonglong2 v0 = ld_rec16(src), v1 = ld_rec16(src + 2);
        k[0] = v0.x; k[1] = v0.y; k[2] = v1.x; k[3] = v1.y;
    } else {
#pragma unroll
        for (int q = 0; q < W; ++q) k[q] = src[q];
    }
}
// a < b for two records of the same first word (the words behind it, from memory)
template <int W>
__device__ __forceinline__ bool rest_less(const u64 *__restrict__ ra, const u64 *__restrict__ rb) {
#pragma unroll
    for (int q = 1; q < W; ++q) { const u64 x = ra[q], y = rb[q]; if (x != y) return x < y; }
    return false;
}

// WARPS x 32 threads; a warp holds U rows of 32 records at a time; TSMAX table slots (power of two), MAXSOLID sort
// places, NB = 1024 bins. Counts are 16-bit halves of u32 words (a segment has at most window + chunk < 65,536 records).
// The records of a segment are dealt to the warps in groups of U full rows (no lane is ever idle there, so the group
// code has no predicates); the rows that do not fill a group and the partial last row go one by one.
template <int W, int WARPS, int MINB, int U, int TSMAX, int MAXSOLID, int CB, bool LIST = false>
__global__ void __launch_bounds__(WARPS * 32, MINB)
hash_count_kernel(HashCountArgs a) {
    static_assert(CB == 2 || CB == 4, "counts are 16-bit halves of u32 words or u32 words");
    constexpr int THREADS = WARPS * 32;
    constexpr bool MW = W > 1;
    constexpr bool REC = W == 2;                         // a.keys holds the records themselves (W words each), no a.vals
    using rep_t = unsigned short;                                               // place of a record inside its segment
    constexpr size_t kOffCnt = (size_t)TSMAX * 8, kOffLKey = kOffCnt + (size_t)TSMAX * CB, kOffLCnt = kOffLKey + (size_t)MAXSOLID * 8;
    constexpr size_t kOffTRep = kOffLCnt + (size_t)MAXSOLID * 4, kOffLRep = kOffTRep + (MW ? (size_t)TSMAX * 2 : 0);
    constexpr size_t kOffSlot = kOffLRep + (MW ? (size_t)MAXSOLID * 2 : 0);     // (W > 1) rep_t[TSMAX]: the slot of each of the first TSMAX records
    extern __shared__ __align__(16) unsigned char smem_raw[];
    u64 *t_key = reinterpret_cast<u64 *>(smem_raw);                             // u64[TSMAX]: key (W = 1) or fingerprint
    u32 *t_cnt = reinterpret_cast<u32 *>(smem_raw + kOffCnt);                   // CB = 2: u16[TSMAX] as u32 pairs; CB = 4: u32[TSMAX]
    u64 *l_key = reinterpret_cast<u64 *>(smem_raw + kOffLKey);                  // u64[MAXSOLID]: first key word
    u32 *l_cnt = reinterpret_cast<u32 *>(smem_raw + kOffLCnt);
    rep_t *t_rep = reinterpret_cast<rep_t *>(smem_raw + kOffTRep);              // (W > 1) rep_t[TSMAX]: who installed the slot
    rep_t *l_rep = reinterpret_cast<rep_t *>(smem_raw + kOffLRep);              // (W > 1) rep_t[MAXSOLID]
    rep_t *s_slot = reinterpret_cast<rep_t *>(smem_raw + kOffSlot);
    __shared__ u32 s_ones, s_full, s_nsolid, s_distinct, s_clash;
    __shared__ u64 s_sum, s_look[2][4], s_krange[2];
    __shared__ u32 s_w[WARPS];
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const u32 tkey_s = (u32)__cvta_generic_to_shared(smem_raw);
    // tickets run over the segments, or over the list of the non-empty ones (long buckets: a third of the nominal segments
    // is empty there, and an iteration without records still costs its barriers and the latency of the look-ahead)
    const u64 nseg = LIST ? (u64)*a.n_list : a.nseg;

    // Tickets are taken two segments ahead by thread 0, which also fetches the bounds of that segment while the CTA works:
    // s_look[p] = {segment, first record, end} of the iteration with parity p (nothing depends on a load it just issued).
    auto bounds_of = [&](u64 t, u64 &id, u64 &bs, u64 &be) {   // ticket t -> segment id and its records [bs, be)
        id = t; bs = be = 0;
        if (t < nseg) { if constexpr (LIST) id = a.seg_list[t]; bs = a.seg_start[id]; be = a.seg_start[id + 1]; }
    };
    if (tid == 0) {
        const u64 t0 = atomicAdd(a.ticket, 1u), t1 = atomicAdd(a.ticket, 1u);
        u64 i0, b0, e0, i1, b1, e1;
        bounds_of(t0, i0, b0, e0); bounds_of(t1, i1, b1, e1);
        s_look[0][0] = t0; s_look[0][1] = b0; s_look[0][2] = e0; s_look[0][3] = i0;
        s_look[1][0] = t1; s_look[1][1] = b1; s_look[1][2] = e1; s_look[1][3] = i1;
    }
    __syncthreads();
    u64 seg = s_look[0][0];                              // the ticket; seg_id is the segment
    if (seg >= nseg) return;
    u64 s = s_look[0][1], e = s_look[0][2], seg_id = s_look[0][3];
    // full groups of the segment [bs, be) (none for the segment that ends with the last record of all: it alone can hold
    // the all-ones key, which is counted beside the table by the row-by-row code)
    auto groups_of = [&](u64 bs, u64 be) { return be <= bs || be == a.n ? 0u : ((u32)(be - bs) >> 5) / (u32)U; };
    u64 cur[U][1];
    u32 cur_v[U];                                        // (W > 1) the record indices of the rows in cur
    auto load_group_v = [&](u64 (&k)[U][1], u32 (&v)[U], u64 first) {   // rows first + 32 u + lane of keys (and vals)
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if constexpr (REC) {
                u64 rec[W];
                load_key<W>(a.keys + (first + 32 * u + lane) * W, rec);
                k[u][0] = pair_key<W>(rec, 0u, a.weak_fp);
                v[u] = 0;
            } else {
                k[u][0] = ld_stream(a.keys + first + 32 * u + lane);
                if constexpr (MW) v[u] = a.vals[first + 32 * u + lane]; else v[u] = 0;
            }
        }
    };
    // src = a.keys + (index of the first key): the index is what counts (records of W words in REC mode)
    auto load_group = [&](u64 (&k)[U][1], const u64 *src) { load_group_v(k, cur_v, (u64)(src - a.keys)); };
    // the stand-in of the i-th key of the segment that starts at s0, from memory
    auto key_at = [&](u64 s0, u32 i) -> u64 {
        if constexpr (REC) { u64 rec[W]; load_key<W>(a.keys + (s0 + i) * W, rec); return pair_key<W>(rec, 0u, a.weak_fp); }
        else return ld_stream(a.keys + s0 + i);
    };
    // (W > 1) the record of the i-th key of the segment that starts at s0
    auto rec_of = [&](u64 s0, u32 i) -> const u64 * {
        if constexpr (REC) return a.keys + (s0 + i) * W; else return a.recs + (size_t)a.vals[s0 + i] * W;
    };
    // (W > 1) a key that met its slot taken will be compared with the record that installed it: its own record is asked
    // for now (into L2), while the rest of the segment is inserted
    auto want_rec = [&](u32 v) {
        if constexpr (!REC) asm volatile("prefetch.global.L2 [%0];" ::"l"(a.recs + (size_t)v * W));
    };
    if (warp < groups_of(s, e)) load_group(cur, a.keys + s + (u64)warp * (32 * U));

    for (u32 it = 0;; ++it) {
        const u32 m = e > s ? (u32)(e - s) : 0u;         // a segment has fewer than 2^16 records
        // table size: the power of two from 1.5 x the records of the segment on (all of them might be distinct)
        u32 TS = 1024;
        while (TS < (u32)TSMAX && (u64)TS * 2 < (u64)m * 3) TS <<= 1;
        const u32 mask8 = (TS - 1u) << 3, hshift = 32u - (u32)__ffs(TS) + 1u;
        {
            uint4 *k4 = reinterpret_cast<uint4 *>(t_key), *c4 = reinterpret_cast<uint4 *>(t_cnt);
            const uint4 ones = make_uint4(~0u, ~0u, ~0u, ~0u), zero = make_uint4(0u, 0u, 0u, 0u);
            for (u32 i = tid; i < TS / 2; i += THREADS) k4[i] = ones;
            for (u32 i = tid; i < TS * CB / 16; i += THREADS) c4[i] = zero;
        }
        u64 la_seg = 0, la_s = 0, la_e = 0, la_id = 0;   // (thread 0) the segment of the iteration after the next one
        u64 kf = 0, kl = 0;                              // (thread 32) first word of the first and of the last record
        if (tid == 0) {
            s_ones = 0; s_full = 0; s_nsolid = 0; s_distinct = 0; s_sum = 0; s_clash = 0;
            la_seg = atomicAdd(a.ticket, 1u);          // consumed behind the insert phase: nothing waits for it here
            // the keys of my NEXT segment (its bounds came an iteration ago) are asked for now, into L2, by the TMA unit: the
            // loads of its insert phase, half of which are issued just before they are needed, then come from there
            const u64 pn_s = s_look[(it + 1) & 1][1], pn_e = s_look[(it + 1) & 1][2];
            if (pn_e > pn_s) {
                constexpr u64 KW = REC ? W : 1;
                const u64 p0 = (u64)(a.keys + pn_s * KW) & ~15ull, p1 = ((u64)(a.keys + pn_e * KW) + 15ull) & ~15ull;
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p0), "r"((u32)(p1 - p0)) : "memory");
            }
        }
        if (tid == 32 % THREADS && m) { kf = a.keys[s * (REC ? W : 1)]; kl = a.keys[(e - 1) * (REC ? W : 1)]; }   // first words
        __syncthreads();

        // ---- 1: insert ---------------------------------------------------------------------------------------------------
        u32 created = 0;
        const bool last_seg = e == a.n;
        // count of the slot at byte offset a8 of the key table (CB = 2: 16-bit halves, two slots per word)
        auto cnt_add = [&](u32 a8) {
            if constexpr (CB == 2) s_red_add<TSMAX * 8>(tkey_s + ((a8 >> 2) & ~3u), (a8 & 8u) ? 0x10000u : 1u);
            else s_red_add<TSMAX * 8>(tkey_s + (a8 >> 1), 1u);
        };
        // NR rows held by the warp (row r = records i0 + 32 r + lane of the segment): first the home slot of every record
        // (one CAS that installs the key or returns what is there, no loop), then ONE probing loop for the records whose
        // home slot holds another key
        auto insert_rows = [&](auto nr_tag, const u64 (*k)[1], const u32 *kv, u32 i0, bool valid) {
            constexpr int NR = decltype(nr_tag)::value;
            u64 old[NR], f[NR]; u32 a8[NR];
#pragma unroll
            for (int r = 0; r < NR; ++r) {
                f[r] = k[r][0];
                a8[r] = hash_slot(f[r], hshift) << 3;
                old[r] = f[r];
                if (NR > 1 || valid) old[r] = s_cas64(tkey_s + a8[r], kEmpty, f[r]);
            }
            u32 pend = 0;
#pragma unroll
            for (int r = 0; r < NR; ++r) {
                const bool emp = old[r] == kEmpty;
                if (NR > 1 || valid) {
                    if (emp || old[r] == f[r]) cnt_add(a8[r]); else pend |= 1u << r;
                    if constexpr (MW) {
                        const u32 idx = i0 + 32u * (u32)r + lane;
                        if (emp) t_rep[a8[r] >> 3] = (rep_t)idx;
                        if (idx < (u32)TSMAX && (emp || old[r] == f[r])) s_slot[idx] = (rep_t)(a8[r] >> 3);
                        if (!emp) want_rec(kv[r]);     // a copy, or a key that goes on probing (most of those end as copies)
                    }
                    created += emp;
                }
            }
            if (pend) {
                u64 key = 0; u32 b8 = 0, probes = 0, who = 0;
                bool have = false;
                for (;;) {
                    if (!have) {
                        if (!pend) break;
                        const u32 r = (u32)__ffs(pend) - 1u;
                        pend &= pend - 1u;
                        key = f[0]; b8 = a8[0];
#pragma unroll
                        for (int q = 1; q < NR; ++q) if (r == (u32)q) { key = f[q]; b8 = a8[q]; }
                        who = i0 + 32u * r + lane;
                        probes = 0; have = true;
                    }
                    b8 = (b8 + 8u) & mask8;
                    const u64 o = s_cas64(tkey_s + b8, kEmpty, key);
                    if (o == kEmpty || o == key) {
                        cnt_add(b8); created += o == kEmpty; have = false;
                        if constexpr (MW) {
                            if (o == kEmpty) t_rep[b8 >> 3] = (rep_t)who;
                            if (who < (u32)TSMAX) s_slot[who] = (rep_t)(b8 >> 3);
                        }
                    } else if (++probes >= TS) { s_full = 1; have = false; }
                }
            }
        };
        const u32 G = groups_of(s, e);
        {
            u64 nxt[U][1];
            u32 nxt_v[U];
            for (u32 g = warp; g < G; g += 2 * WARPS) {  // two groups per round: one is inserted while the other arrives
                const bool more = g + WARPS < G;
                if (more) load_group_v(nxt, nxt_v, s + (u64)(g + WARPS) * (32 * U));
                insert_rows(std::integral_constant<int, U>{}, cur, cur_v, g * (32u * U), true);
                if (g + 2 * WARPS < G) load_group(cur, a.keys + s + (u64)(g + 2 * WARPS) * (32 * U));
                if (more) insert_rows(std::integral_constant<int, U>{}, nxt, nxt_v, (g + WARPS) * (32u * U), true);
            }
        }
        {   // the rows behind the last full group, and the partial last row: x-th of them belongs to warp (G + x) % WARPS
            const u32 row0 = G * (u32)U, nx = ((m + 31u) >> 5) - row0;
            for (u32 x = (warp + WARPS - G % WARPS) % WARPS; x < nx; x += WARPS) {
                const u32 i = (row0 + x) * 32u + lane;
                const bool valid = i < m;
                u64 key[1][1];
                u32 kv[1];
                key[0][0] = valid ? key_at(s, i) : 0ull;
                kv[0] = (MW && !REC && valid) ? a.vals[s + i] : 0u;
                if (!MW && last_seg && valid && key[0][0] == kEmpty) { atomicAdd(&s_ones, 1u); insert_rows(std::integral_constant<int, 1>{}, key, kv, (row0 + x) * 32u, false); }
                else insert_rows(std::integral_constant<int, 1>{}, key, kv, (row0 + x) * 32u, valid);
            }
        }
        // the first records of my next segment are on their way while this one is finished (its bounds came an iteration ago)
        const u64 next = s_look[(it + 1) & 1][0], ns_ = s_look[(it + 1) & 1][1], ne_ = s_look[(it + 1) & 1][2], nid_ = s_look[(it + 1) & 1][3];
        if (!MW && next < nseg && warp < groups_of(ns_, ne_)) load_group(cur, a.keys + ns_ + (u64)warp * (32 * U));
        if (created) atomicAdd(&s_distinct, created);
        if (tid == 32 % THREADS) { s_krange[0] = kf >> a.top_shift; s_krange[1] = kl >> a.top_shift; }
        __syncthreads();
        if (tid == 0) bounds_of(la_seg, la_id, la_s, la_e);   // stored at the end of the iteration
        const u64 kfirst = s_krange[0], klast = s_krange[1];
        const bool full = s_full != 0;
        if (full && tid == 0) atomicOr(a.overflow, 2u);

        // ---- 1b (W > 1): every record against the one that installed its slot -------------------------------------------------------
        if constexpr (MW) {
            if (!full) {
                // four keys per thread and round, so that the reads through the indices (two dependent loads per record,
                // two records per check) of a round are in flight together
                constexpr int VB = 4;
                for (u32 i0 = tid; i0 < m; i0 += VB * THREADS) {
                    u32 rep[VB], need = 0;
#pragma unroll
                    for (int u = 0; u < VB; ++u) {
                        const u32 i = i0 + (u32)u * THREADS;
                        rep[u] = i;
                        if (i < m) {
                            u32 slot;
                            if (i < (u32)TSMAX) slot = s_slot[i];   // noted when the key was inserted
                            else {
                                const u64 f = key_at(s, i);
                                u32 b8 = hash_slot(f, hshift) << 3;
                                while (t_key[b8 >> 3] != f) b8 = (b8 + 8u) & mask8;   // it is there: the table was not full
                                slot = b8 >> 3;
                            }
                            rep[u] = t_rep[slot];
                            need |= (rep[u] != i ? 1u : 0u) << u;
                        }
                    }
                    if (need == 0) continue;
                    u32 vi[VB], vr[VB];
#pragma unroll
                    for (int u = 0; u < VB; ++u) {
                        vi[u] = 0; vr[u] = 0;
                        if constexpr (!REC) {
                            if ((need >> u) & 1u) { vi[u] = a.vals[s + i0 + (u32)u * THREADS]; vr[u] = a.vals[s + rep[u]]; }
                        }
                    }
                    bool same = true;
#pragma unroll
                    for (int u = 0; u < VB; ++u) {
                        if ((need >> u) & 1u) {
                            u64 k[W], o[W];
                            if constexpr (REC) {
                                load_key<W>(a.keys + (s + i0 + (u32)u * THREADS) * W, k);
                                load_key<W>(a.keys + (s + rep[u]) * W, o);
                            } else {
                                load_key<W>(a.recs + (size_t)vi[u] * W, k);
                                load_key<W>(a.recs + (size_t)vr[u] * W, o);
                            }
#pragma unroll
                            for (int q = 0; q < W; ++q) same = same && o[q] == k[q];
                        }
                    }
                    if (!same) s_clash = 1;
                }
            }
            if (next < nseg && warp < groups_of(ns_, ne_)) load_group(cur, a.keys + ns_ + (u64)warp * (32 * U));
            // no barrier here: the check only reads the table, and so does the scan that follows; a warp that had little to
            // check goes on. A mismatch is reported behind the next barrier; until then the segment is handled as usual
            // (its sizes are sound, its content is discarded with everything else when the flag is set)
        }

        // ---- 2: the solid slots, compacted to this iteration's list ------------------------------------------------------------
        u64 sum = 0;
        if (!full && m) {   // the live part of the table, 16 bytes of counts (8 or 4 slots) per load; most vectors hold no solid edge
            const uint4 *c4 = reinterpret_cast<const uint4 *>(t_cnt);
            const u32 d = a.d;
            constexpr u32 SPV = 16 / CB;                 // slots per vector
            for (u32 v = tid; v < TS / SPV; v += THREADS) {
                const uint4 w = c4[v];
                if (d == 2 && ((w.x | w.y | w.z | w.w) & (CB == 2 ? 0xfffefffeu : 0xfffffffeu)) == 0) continue;   // no count above 1
                const u32 wd[4] = {w.x, w.y, w.z, w.w};
                u32 mq = 0;                              // bit q: slot SPV v + q holds a solid edge
#pragma unroll
                for (u32 q = 0; q < 4; ++q) {
                    if constexpr (CB == 2) mq |= ((wd[q] & 0xffffu) >= d ? 1u : 0u) << (2 * q) | ((wd[q] >> 16) >= d ? 2u : 0u) << (2 * q);
                    else mq |= (wd[q] >= d ? 1u : 0u) << q;
                }
                while (mq) {
                    const u32 q = (u32)__ffs(mq) - 1u;
                    mq &= mq - 1u;
                    const u32 wi = CB == 2 ? q >> 1 : q;
                    u32 wq = wd[0];
                    if (wi == 1) wq = wd[1];
                    if (wi == 2) wq = wd[2];
                    if (wi == 3) wq = wd[3];
                    const u32 c = CB == 2 ? (wq >> ((q & 1u) * 16u)) & 0xffffu : wq;
                    const u32 p = atomicAdd(&s_nsolid, 1u);
                    if (p < (u32)MAXSOLID) {
                        if constexpr (MW) { const u32 rep = t_rep[v * SPV + q]; l_rep[p] = (rep_t)rep; l_key[p] = rec_of(s, rep)[0]; }
                        else l_key[p] = t_key[v * SPV + q];
                        l_cnt[p] = c;
                    }
                    sum += c;
                }
            }
            if (tid == 0 && s_ones) {
                atomicAdd(&s_distinct, 1u);
                if (s_ones >= a.d) {
                    const u32 p = atomicAdd(&s_nsolid, 1u);
                    if (p < (u32)MAXSOLID) { l_key[p] = kEmpty; l_cnt[p] = s_ones; }
                    sum += s_ones;
                }
            }
            sum = warp_reduce_add64(sum);
            if (lane == 0 && sum) atomicAdd(&s_sum, sum);
        }
        __syncthreads();
        if constexpr (MW) { if (tid == 0 && s_clash) atomicOr(a.overflow, 16u); }
        u32 ns = s_nsolid;
        if (ns > (u32)MAXSOLID) { if (tid == 0) atomicOr(a.overflow, 4u); ns = 0; }
        if (full) ns = 0;
        // ---- 3a: the count of the segment, the sum of its block, statistics ---------------------------------------------------------
        if (tid == 0) {
            a.seg_count[seg_id] = ns;
            if (ns) atomicAdd(a.blk_sum + seg_id / kSegBlock, (u64)ns);
            u64 *slot = a.stat_slots + (size_t)(seg_id & (kStatSlots - 1)) * kStatSlotWords;
            if (ns) atomicAdd(&slot[1], s_sum);
            if (s_distinct && !full) atomicAdd(&slot[0], (u64)s_distinct);
        }

        // ---- 3b: order the list by key. The solid edges of a segment are spread evenly over its key range, so one pass of
        //          order-preserving binning (1,024 bins over the range of the segment's buckets) leaves bins of one or two
        //          entries, which the owner of the bin puts in order by insertion. The table is dead: bins and the ordered
        //          entries live in its place. ---------------------------------------------------------------------------------------
        constexpr int NB = 1024, Q = NB / THREADS, QE = MAXSOLID / THREADS;   // bins per thread; list entries per thread
        static_assert(NB % THREADS == 0 && MAXSOLID % THREADS == 0 && (size_t)NB * 4 <= (size_t)TSMAX * CB && (size_t)MAXSOLID * 14 <= (size_t)TSMAX * 8, "layout");
        if (ns) {
            u32 *bins = t_cnt;
            u64 *o_key = t_key;
            u32 *o_cnt = reinterpret_cast<u32 *>(t_key + MAXSOLID);
            rep_t *o_rep = reinterpret_cast<rep_t *>(o_cnt + MAXSOLID);
            const u64 k0 = kfirst << a.top_shift;
            const u64 rm1 = ((klast - kfirst + 1ull) << a.top_shift) - 1ull;  // largest offset inside the segment's buckets
            const int sh0 = 54 - __clzll((long long)rm1), sh = sh0 > 0 ? sh0 : 0;   // (rm1 >> sh) < 1024
#pragma unroll
            for (int q = 0; q < Q; ++q) bins[tid + q * THREADS] = 0;
            __syncthreads();
            u32 myb[QE], myr[QE];
#pragma unroll
            for (int q = 0; q < QE; ++q) {
                const u32 i = tid + q * THREADS;
                myb[q] = 0; myr[q] = 0;
                if (i < ns) { myb[q] = (u32)((l_key[i] - k0) >> sh); myr[q] = atomicAdd(&bins[myb[q]], 1u); }
            }
            __syncthreads();
            u32 c[Q], csum = 0;
#pragma unroll
            for (int q = 0; q < Q; ++q) { c[q] = bins[Q * tid + q]; csum += c[q]; }
            const u32 incl = warp_incl_scan_add(csum);
            if (lane == 31u) s_w[warp] = incl;
            __syncthreads();
            u32 base0 = incl - csum;
            for (u32 w = 0; w < warp; ++w) base0 += s_w[w];
            {
                u32 run = base0;
#pragma unroll
                for (int q = 0; q < Q; ++q) { bins[Q * tid + q] = run; run += c[q]; }
            }
            __syncthreads();
#pragma unroll
            for (int q = 0; q < QE; ++q) {
                const u32 i = tid + q * THREADS;
                if (i < ns) {
                    const u32 p = bins[myb[q]] + myr[q];
                    o_key[p] = l_key[i]; o_cnt[p] = l_cnt[i];
                    if constexpr (MW) o_rep[p] = l_rep[i];
                }
            }
            __syncthreads();
            {
                u32 b0 = base0;
#pragma unroll
                for (int q = 0; q < Q; ++q) {
                    for (u32 x = 1; x < c[q]; ++x) {                           // insertion sort of places [b0, b0 + c)
                        const u64 kx = o_key[b0 + x]; const u32 cx = o_cnt[b0 + x];
                        const u32 rx = MW ? o_rep[b0 + x] : 0u;
                        u32 y = x;
                        while (y > 0) {
                            const u64 ky = o_key[b0 + y - 1];
                            bool gt = ky > kx;           // entry y - 1 > entry x
                            if constexpr (MW) { if (ky == kx) gt = rest_less<W>(rec_of(s, rx), rec_of(s, o_rep[b0 + y - 1])); }
                            if (!gt) break;
                            o_key[b0 + y] = ky; o_cnt[b0 + y] = o_cnt[b0 + y - 1];
                            if constexpr (MW) o_rep[b0 + y] = o_rep[b0 + y - 1];
                            --y;
                        }
                        o_key[b0 + y] = kx; o_cnt[b0 + y] = cx;
                        if constexpr (MW) o_rep[b0 + y] = (rep_t)rx;
                    }
                    b0 += c[q];
                }
            }
            __syncthreads();
            // staging (8 W bytes per record, the sorter's spare buffer): the segment owns places [s, e); its ns <= (e - s) / d
            // solid keys (d >= 2) fill the first half at most, their u32 counts start at the middle place
            u32 *stage_cnt = reinterpret_cast<u32 *>(a.stage_keys + (s + ((m + 1u) >> 1)) * W);
            for (u32 i = tid; i < ns; i += THREADS) {
                if constexpr (MW) {
                    u64 k[W];
                    load_key<W>(rec_of(s, o_rep[i]), k);
#pragma unroll
                    for (int q = 0; q < W; ++q) a.stage_keys[(s + i) * W + q] = k[q];
                } else a.stage_keys[s + i] = o_key[i];
                stage_cnt[i] = o_cnt[i];
            }
        }
        if (next >= nseg) break;
        if (tid == 0) { s_look[it & 1][0] = la_seg; s_look[it & 1][1] = la_s; s_look[it & 1][2] = la_e; s_look[it & 1][3] = la_id; }
        seg = next; s = ns_; e = ne_; seg_id = nid_;
        __syncthreads();   // the table is cleared next
    }
}

// seg_list[0 .. *n_list) = the segments with records (long buckets only). Nearly in order: a warp appends the non-empty ones
// of its 32 segments at a place taken from *n_list; the order in which segments are counted is free (every segment writes
// to its own places).
__global__ void __launch_bounds__(256) hash_list_kernel(const u64 *__restrict__ seg_start, u64 nseg, u32 *__restrict__ seg_list, u32 *n_list) {
    const u64 c = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    const bool has = c < nseg && seg_start[c] < seg_start[c + 1];
    const u32 b = __ballot_sync(0xffffffffu, has);
    if (b == 0) return;
    u32 base = 0;
    if (lane_id() == 0) base = atomicAdd(n_list, (u32)__popc(b));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (has) seg_list[base + (u32)__popc(b & lanemask_lt())] = (u32)c;
}

// blk_sum[b] (solid edges of segments [64 b, 64 b + 64)) -> exclusive prefix in place, total to *total and the output
// cursor behind this range; one block (a range of 2^34 records has at most 2^17 blocks of 64 segments of 2,048 records)
__global__ void __launch_bounds__(1024) hash_scan_kernel(u64 *__restrict__ blk_sum, u64 nblk, u64 *total, const u64 *cursor_in, u64 *cursor_out) {
    __shared__ u64 s_w[32];
    __shared__ u64 s_carry;
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (u64 base = 0; base < nblk; base += 1024) {
        const u64 i = base + tid;
        const u64 v = i < nblk ? blk_sum[i] : 0;
        u64 incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            u64 t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= (u32)o) incl += t;
        }
        if (lane == 31) s_w[warp] = incl;
        __syncthreads();
        u64 off = s_carry;
        for (u32 w = 0; w < warp; ++w) off += s_w[w];
        if (i < nblk) blk_sum[i] = off + incl - v;
        __syncthreads();
        if (tid == 1023) s_carry = off + incl;
        __syncthreads();
    }
    if (tid == 0) { *total = s_carry; *cursor_out = *cursor_in + s_carry; }
}

// the staged solid edges of every segment appended to the output, in segment (= key) order: a CTA per block of 64
// segments (prefix of their counts in shared memory), a warp per segment
__global__ void __launch_bounds__(256) hash_copy_kernel(HashCountArgs a) {
    __shared__ u64 s_off[kSegBlock];
    __shared__ u64 s_w[kSegBlock / 32];
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const u64 base = *a.cursor_in;
    for (u64 blk = blockIdx.x; blk * kSegBlock < a.nseg; blk += gridDim.x) {
        u64 v = 0, incl = 0;
        if (tid < kSegBlock) {
            const u64 seg0 = blk * kSegBlock + tid;
            v = seg0 < a.nseg ? a.seg_count[seg0] : 0;
            incl = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                u64 t = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= (u32)o) incl += t;
            }
            if (lane == 31) s_w[warp] = incl;
        }
        __syncthreads();
        if (tid < kSegBlock) {
            u64 off = a.blk_sum[blk];
            for (u32 w = 0; w < warp; ++w) off += s_w[w];
            s_off[tid] = off + incl - v;
        }
        __syncthreads();
        for (u32 j = warp; j < kSegBlock; j += 8) {
            const u64 seg = blk * kSegBlock + j;
            if (seg >= a.nseg) break;
            const u64 cnt = a.seg_count[seg];
            if (cnt == 0) continue;
            const u64 s = a.seg_start[seg], e = a.seg_start[seg + 1];
            const u32 W = a.W ? a.W : 1u;
            const u32 *stage_cnt = reinterpret_cast<const u32 *>(a.stage_keys + (s + ((e - s + 1) >> 1)) * W);
            const u64 pos0 = base + s_off[j];
            const u64 room = pos0 < a.out_cap ? a.out_cap - pos0 : 0, take = cnt < room ? cnt : room;
            for (u64 i = lane; i < take * W; i += 32) a.out_keys[pos0 * W + i] = a.stage_keys[s * W + i];
            for (u64 i = lane; i < take; i += 32) a.out_mult[pos0 + i] = stage_cnt[i];
        }
        __syncthreads();
    }
}

// shapes: long buckets (chunk 4,096: one or two buckets per segment) and short ones (chunk 2,048: many buckets per segment)
template <int W, int WARPS, int MINB, int U, int TSMAX, int MAXSOLID, int CB, bool LIST = false>
struct HashShape {
    static constexpr int THREADS = WARPS * 32;
    static constexpr size_t kSmem = (size_t)TSMAX * (8 + CB) + (size_t)MAXSOLID * 12 + (W > 1 ? (size_t)TSMAX * 4 + (size_t)MAXSOLID * 2 : 0);
    static int setup(int *blocks_per_sm) {
        int e = (int)cudaFuncSetAttribute(hash_count_kernel<W, WARPS, MINB, U, TSMAX, MAXSOLID, CB, LIST>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem);
        if (e) return e;
        return (int)cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, hash_count_kernel<W, WARPS, MINB, U, TSMAX, MAXSOLID, CB, LIST>, THREADS, kSmem);
    }
    static int launch(const HashCountArgs &a, int blocks_per_sm, cudaStream_t s) {
        u64 g = (u64)num_sms() * (u64)(blocks_per_sm > 0 ? blocks_per_sm : 1);
        if (g > a.nseg) g = a.nseg;
        hash_count_kernel<W, WARPS, MINB, U, TSMAX, MAXSOLID, CB, LIST><<<(unsigned)g, THREADS, kSmem, s>>>(a);
        return (int)cudaGetLastError();
    }
};
#ifndef SDBG_HASH_BIG_TS
#define SDBG_HASH_BIG_TS 8192
#endif
#ifndef SDBG_HASH_BIG_CB
#define SDBG_HASH_BIG_CB 4
#endif
#ifndef SDBG_BIG_U
#define SDBG_BIG_U 4
#endif
#ifndef SDBG_SMALL_U
#define SDBG_SMALL_U 4
#endif
#ifndef SDBG_HASH_BIG
#define SDBG_HASH_BIG 16, 2, SDBG_BIG_U, SDBG_HASH_BIG_TS, 1024, SDBG_HASH_BIG_CB
#endif
#ifndef SDBG_HASH_SMALL
#define SDBG_HASH_SMALL 8, 4, SDBG_SMALL_U, 4096, 1024, 2
#endif
#ifndef SDBG_MW_WARPS
#define SDBG_MW_WARPS 8
#define SDBG_MW_MINB 3
#define SDBG_MW_U 4
#endif
#ifndef SDBG_HASH_MW   // keys of several words (one-word stand-ins with an index payload): short buckets only
#define SDBG_HASH_MW SDBG_MW_WARPS, SDBG_MW_MINB, SDBG_MW_U, 4096, 1024, 2
#endif
using HashBig = HashShape<1, SDBG_HASH_BIG, true>;       // always over the list of the non-empty segments
using HashSmall = HashShape<1, SDBG_HASH_SMALL>;
using HashMW2 = HashShape<2, SDBG_HASH_MW>;
using HashMW3 = HashShape<3, SDBG_HASH_MW>;
using HashMW4 = HashShape<4, SDBG_HASH_MW>;
static int g_occ_big = 0, g_occ_small = 0, g_occ_mw[5] = {0, 0, 0, 0, 0};

int hash_setup() {
    int e = HashBig::setup(&g_occ_big);
    if (e) return e;
    if ((e = HashMW2::setup(&g_occ_mw[2]))) return e;
    if ((e = HashMW3::setup(&g_occ_mw[3]))) return e;
    if ((e = HashMW4::setup(&g_occ_mw[4]))) return e;
    return HashSmall::setup(&g_occ_small);
}

void launch_hash_bounds(const HashCountArgs &a, cudaStream_t s) {
    const u64 warps = a.nseg + 1, blocks = (warps + 7) / 8;
    if (a.seg_list) cudaMemsetAsync(a.seg_count, 0, a.nseg * 8, s);   // the empty segments are never visited
    hash_bounds_kernel<<<(unsigned)blocks, 256, 0, s>>>(a.keys, a.W == 2 ? 2u : 1u, a.n, a.top_shift, a.chunk, a.window, a.nseg, a.seg_start, a.overflow);
    if (a.seg_list) hash_list_kernel<<<(unsigned)((a.nseg + 255) / 256), 256, 0, s>>>(a.seg_start, a.nseg, a.seg_list, a.n_list);
}
int launch_hash_count(const HashCountArgs &a, cudaStream_t s) {
    if (a.nseg == 0 || a.nseg > 0x7fffffffull || (u64)a.window + a.chunk >= 65536) return (int)cudaErrorInvalidValue;
    if (a.W > 1) {                                       // several words per key: the short-bucket shape only
        if (a.chunk > 2048) return (int)cudaErrorInvalidValue;
        switch (a.W) {
            case 2: return HashMW2::launch(a, g_occ_mw[2], s);
            case 3: return HashMW3::launch(a, g_occ_mw[3], s);
            case 4: return HashMW4::launch(a, g_occ_mw[4], s);
        }
        return (int)cudaErrorInvalidValue;
    }
    if (a.chunk >= 4096) return a.seg_list ? HashBig::launch(a, g_occ_big, s) : (int)cudaErrorInvalidValue;
    return a.seg_list ? (int)cudaErrorInvalidValue : HashSmall::launch(a, g_occ_small, s);
}
void launch_hash_append(const HashCountArgs &a, u64 *total, cudaStream_t s) {
    const u64 nblk = (a.nseg + kSegBlock - 1) / kSegBlock;
    hash_scan_kernel<<<1, 1024, 0, s>>>(a.blk_sum, nblk, total, a.cursor_in, a.cursor_out);
    const u64 cap = (u64)num_sms() * 8;
    hash_copy_kernel<<<(unsigned)(nblk < cap ? nblk : cap), 256, 0, s>>>(a);
}

}  // namespace sdbg

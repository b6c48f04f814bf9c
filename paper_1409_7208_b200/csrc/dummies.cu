// dummies.cu — the lossless extras of the SdBG (readings A18-A20 of DESIGN.md):
// "a bit-vector of length m to mark the validity of each edge ... and an auxiliary vector of 2kt bits (where k is the
// k-mer size and t is the number of zero-indegree vertices) to store the sequence of zero-indegree vertices", plus the
// outgoing `$` edges of Bowe et al. for the nodes that have no outgoing edge.
//
// Over the sorted solid edges S: src(e) = e[0..k) is the top 2k bits of the key; tgt(e) = e[1..k] as a colex node key
// is (e[k], e[k-1], ..., e[1]) = the key shifted right by one symbol with its last symbol put in front. The target
// keys are sorted with the same radix sorter; then
//   Z_out = tgt(S) \ src(S)  (binary search of every distinct target in the edge list)   -> one `$` edge per node
//   Z_in  = src(S) \ tgt(S)  (binary search of every node of the edge list in the targets) -> auxiliary vector
// and the final arrays are the emitted arrays of S with the `$` edges merged in by node order (a `$` edge changes no
// flag of a real edge: it has a node of its own and no outgoing base), written one output position per thread.
#include "kernels.cuh"

namespace sdbg {

template <int W>
__device__ __forceinline__ void ld_rec(const u64 *__restrict__ a, u64 i, u64 (&k)[W]) {
#pragma unroll
    for (int q = 0; q < W; ++q) k[q] = a[i * W + q];
}

// node (top 2k bits) of a W-word edge key against a WT-word node key: -1, 0, +1
template <int W, int WT>
__device__ __forceinline__ int node_cmp(const u64 (&edge)[W], const u64 (&node)[WT], u32 k) {
#pragma unroll
    for (int q = 0; q < WT; ++q) {
        const int rem = (int)(2 * k) - 64 * q;                       // node bits in this word (> 0 for q < WT)
        const u64 mask = rem >= 64 ? ~0ull : ~0ull << (64 - rem);
        const u64 a = edge[q] & mask, b = node[q];
        if (a != b) return a < b ? -1 : 1;
    }
    return 0;
}

// tgt(e) of every edge as a node key of WT = ceil(2k/64) words
template <int W, int WT>
__global__ void __launch_bounds__(256) target_keys_kernel(const u64 *__restrict__ keys, u64 n, u32 k, u64 *__restrict__ out) {
    const u32 pad = 64u * W - 2u * (k + 1u);
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (u64)gridDim.x * blockDim.x) {
        u64 e[W], t[W];
        ld_rec<W>(keys, i, e);
        const u64 last_sym = (e[W - 1] >> pad) & 3ull;
#pragma unroll
        for (int q = 0; q < W; ++q) t[q] = (e[q] >> 2) | (q ? e[q - 1] << 62 : 0ull);
        t[0] |= last_sym << 62;
#pragma unroll
        for (int q = 0; q < WT; ++q) {
            const int rem = (int)(2 * k) - 64 * q;
            out[i * WT + q] = t[q] & (rem >= 64 ? ~0ull : ~0ull << (64 - rem));
        }
    }
}

// Prefix index over a sorted key list (records of `stride` words): idx[b] = first record whose top pb bits are >= b, for
// b = 0 .. 2^pb (idx[2^pb] = n). The searches below start inside one bucket (a few hundred records for 2^20 buckets)
// instead of the whole list: ~9 steps over neighbouring lines instead of ~28 over gigabytes.
__global__ void __launch_bounds__(256) prefix_index_kernel(const u64 *__restrict__ a, u64 n, u32 stride, u32 pb, u32 *__restrict__ idx) {
    const u64 b = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (b > (1ull << pb)) return;
    u64 lo = 0, hi = n;
    if (b == (1ull << pb)) lo = n;
    else
        while (lo < hi) {
            const u64 mid = lo + ((hi - lo) >> 1);
            if ((a[mid * stride] >> (64 - pb)) < b) lo = mid + 1; else hi = mid;
        }
    idx[b] = (u32)lo;
}

// flag_out[j] = tk[j] is the first of its value and no edge has it as its node; tk sorted
template <int W, int WT>
__global__ void __launch_bounds__(256) flag_zero_out_kernel(const u64 *__restrict__ tk, u64 n, const u64 *__restrict__ keys, u32 k,
                                                            const u32 *__restrict__ idx_edges, u32 pb, uint8_t *__restrict__ flag) {
    for (u64 j = (u64)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += (u64)gridDim.x * blockDim.x) {
        u64 v[WT];
        ld_rec<WT>(tk, j, v);
        bool head = j == 0;
        if (!head) {
            u64 p[WT];
            ld_rec<WT>(tk, j - 1, p);
#pragma unroll
            for (int q = 0; q < WT; ++q) head = head || p[q] != v[q];
        }
        bool is_src = false;
        if (head) {
            const u64 b = v[0] >> (64 - pb);
            u64 lo = idx_edges[b], hi = idx_edges[b + 1];  // first edge whose node is not less than v: inside v's bucket
            const u64 end = hi;
            while (lo < hi) {
                const u64 mid = lo + ((hi - lo) >> 1);
                u64 e[W];
                ld_rec<W>(keys, mid, e);
                if (node_cmp<W, WT>(e, v, k) < 0) lo = mid + 1; else hi = mid;
            }
            if (lo < end) {
                u64 e[W];
                ld_rec<W>(keys, lo, e);
                is_src = node_cmp<W, WT>(e, v, k) == 0;
            }
        }
        flag[j] = head && !is_src;
    }
}

// flag_in[i] = edge i is the last edge of its node and no target equals that node
template <int W, int WT>
__global__ void __launch_bounds__(256) flag_zero_in_kernel(const u64 *__restrict__ keys, u64 n, const u32 *__restrict__ last_bits32,
                                                           const u64 *__restrict__ tk, u32 k, const u32 *__restrict__ idx_tk, u32 pb,
                                                           uint8_t *__restrict__ flag) {
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (u64)gridDim.x * blockDim.x) {
        bool z = false;
        if ((last_bits32[i >> 5] >> (i & 31)) & 1u) {
            u64 e[W];
            ld_rec<W>(keys, i, e);
            const u64 b = e[0] >> (64 - pb);             // pb <= 2k: only node bits
            u64 lo = idx_tk[b], hi = idx_tk[b + 1];      // first target that is not less than the node: inside its bucket
            const u64 end = hi;
            while (lo < hi) {
                const u64 mid = lo + ((hi - lo) >> 1);
                u64 v[WT];
                ld_rec<WT>(tk, mid, v);
                if (node_cmp<W, WT>(e, v, k) > 0) lo = mid + 1; else hi = mid;
            }
            z = true;
            if (lo < end) {
                u64 v[WT];
                ld_rec<WT>(tk, lo, v);
                z = node_cmp<W, WT>(e, v, k) != 0;
            }
        }
        flag[i] = z;
    }
}

// ---- compaction of a byte flag array into the list of flagged indices (ascending) ------------------------------------
// one warp per 1,024 flags; block sums scanned by one block
constexpr u32 kFlagChunk = 1024;
constexpr int kFlagWarps = 8;

template <bool WRITE>
__global__ void __launch_bounds__(kFlagWarps * 32) flag_chunks_kernel(const uint8_t *__restrict__ flag, u64 n, u64 *sums, u32 *__restrict__ out_idx) {
    __shared__ u32 s_cnt[kFlagWarps];
    const u32 lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const u64 chunk = (u64)blockIdx.x * kFlagWarps + warp, c0 = chunk * kFlagChunk;
    u32 *chunk_sums = reinterpret_cast<u32 *>(sums + gridDim.x);
    u64 pos = 0;
    if (WRITE) {
        pos = sums[blockIdx.x];
        for (u32 w = 0; w < warp; ++w) pos += chunk_sums[(u64)blockIdx.x * kFlagWarps + w];
    }
    u32 cnt = 0;
    for (u32 r = 0; r < kFlagChunk / 32; ++r) {
        const u64 i = c0 + r * 32u + lane;
        const bool f = i < n && flag[i];
        const u32 m = __ballot_sync(0xffffffffu, f);
        if (WRITE && f) out_idx[pos + cnt + __popc(m & lanemask_lt())] = (u32)i;
        cnt += __popc(m);
    }
    if (!WRITE) {
        if (lane == 0) { s_cnt[warp] = cnt; chunk_sums[chunk] = cnt; }
        __syncthreads();
        if (threadIdx.x == 0) {
            u64 v = 0;
            for (int w = 0; w < kFlagWarps; ++w) v += s_cnt[w];
            sums[blockIdx.x] = v;
        }
    }
}

__global__ void __launch_bounds__(1024) flag_scan_kernel(u64 *sums, u32 nblocks, u64 *total_out) {
    __shared__ u64 s_w[32];
    __shared__ u64 s_carry;
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (u32 base = 0; base < nblocks; base += 1024) {
        const u32 i = base + tid;
        const u64 v = i < nblocks ? sums[i] : 0ull;
        u64 incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u64 x = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= (u32)o) incl += x;
        }
        if (lane == 31) s_w[warp] = incl;
        __syncthreads();
        u64 off = s_carry;
        for (u32 w = 0; w < warp; ++w) off += s_w[w];
        if (i < nblocks) sums[i] = off + incl - v;
        __syncthreads();
        if (tid == 1023) s_carry = off + incl;
        __syncthreads();
    }
    if (tid == 0) *total_out = s_carry;
}

u64 flag_scratch_bytes(u64 n) {   // block sums (u64) + chunk sums (u32)
    const u64 chunks = (n + kFlagChunk - 1) / kFlagChunk, blocks = (chunks + kFlagWarps - 1) / kFlagWarps;
    return blocks * 8 + blocks * kFlagWarps * 4 + 64;
}

void launch_compact_flags(const uint8_t *flag, u64 n, u64 *scratch, u32 *out_idx, u64 *total_out, cudaStream_t s) {
    const u64 chunks = (n + kFlagChunk - 1) / kFlagChunk, blocks = (chunks + kFlagWarps - 1) / kFlagWarps;
    if (blocks == 0) { cudaMemsetAsync(total_out, 0, 8, s); return; }
    flag_chunks_kernel<false><<<(unsigned)blocks, kFlagWarps * 32, 0, s>>>(flag, n, scratch, out_idx);
    flag_scan_kernel<<<1, 1024, 0, s>>>(scratch, (u32)blocks, total_out);
    flag_chunks_kernel<true><<<(unsigned)blocks, kFlagWarps * 32, 0, s>>>(flag, n, scratch, out_idx);
}

}  // namespace sdbg

namespace sdbg {

// ---- final arrays: the emitted arrays of the real edges with the `$` edges merged in by node order ------------------------
// A `$` edge j goes behind the real edges whose node is less than its own (never equal: it has no real edge) and behind
// the j dummies before it: dpos[j] = j + lower bound of its node in the edge list, strictly increasing, t entries of
// 4 bytes (L2-resident).
template <int W, int WT>
__global__ void __launch_bounds__(256) dummy_pos_kernel(FullArgs a) {
    for (u64 j = (u64)blockIdx.x * blockDim.x + threadIdx.x; j < a.n_zero_out; j += (u64)gridDim.x * blockDim.x) {
        u64 v[WT];
        ld_rec<WT>(a.tk, a.zout_idx[j], v);
        u64 lo = 0, hi = a.n;
        while (lo < hi) {
            const u64 mid = lo + ((hi - lo) >> 1);
            u64 e[W];
            ld_rec<W>(a.keys, mid, e);
            if (node_cmp<W, WT>(e, v, a.k) < 0) lo = mid + 1; else hi = mid;
        }
        a.dpos[j] = (u32)(j + lo);
    }
}

// One thread per OUTPUT position p, one warp per chunk of 1,024 consecutive positions: a warp-uniform lower bound over
// dpos at the start of the chunk, then the chunk is walked in windows of 32 positions; the (at most 32) dummies inside a
// window come as one coalesced load and a bit mask, which tells every lane whether it is a `$` edge and which real
// edge it holds otherwise, and advances the bound. The last and zin words are assembled by ballots, 32 positions per
// store: no atomic and no memset (every word up to ceil(m/64) u64 words is written, tail bits zero).
constexpr u32 kAsmChunk = 1024;

__global__ void __launch_bounds__(256) assemble_kernel(FullArgs a) {
    const u64 m = a.n + a.n_zero_out, padded = (m + 63) / 64 * 64;
    const u32 lane = threadIdx.x & 31u;
    const u64 n_chunks = (padded + kAsmChunk - 1) / kAsmChunk;
    for (u64 chunk = (u64)blockIdx.x * 8 + (threadIdx.x >> 5); chunk < n_chunks; chunk += (u64)gridDim.x * 8) {
        const u64 c0 = chunk * kAsmChunk;
        u64 lo0 = 0, hi = a.n_zero_out;
        while (lo0 < hi) {
            const u64 mid = lo0 + ((hi - lo0) >> 1);
            if (a.dpos[mid] < c0) lo0 = mid + 1; else hi = mid;
        }
        for (u64 p0 = c0; p0 < c0 + kAsmChunk && p0 < padded; p0 += 32) {
            const u64 p = p0 + lane, jd = lo0 + lane;
            const u64 d = jd < a.n_zero_out ? a.dpos[jd] : ~0ull;
            const u32 dmask = __reduce_or_sync(0xffffffffu, d - p0 < 32 ? 1u << (u32)(d - p0) : 0u);
            bool last = false, zin = false;
            if (p < m) {
                const bool dummy = (dmask >> lane) & 1u;
                const u64 i = p - (lo0 + __popc(dmask & lanemask_lt()));
                uint8_t w = 0;
                u32 mult = 0;
                last = true;                             // a `$` edge is the only edge of its node
                if (!dummy) {
                    w = a.W_real[i];
                    mult = a.mult_in[i];
                    last = (a.last_real32[i >> 5] >> (i & 31)) & 1u;
                    zin = a.flag_in[i] != 0;
                }
                a.out_W[p] = w;
                a.out_mult[p] = mult;
            }
            const u32 lw = __ballot_sync(0xffffffffu, last), zw = __ballot_sync(0xffffffffu, zin);
            if (lane == 0) {
                a.out_last32[p0 >> 5] = lw;
                if (a.out_zin32) a.out_zin32[p0 >> 5] = zw;
            }
            lo0 += __popc(dmask);
        }
    }
}

// F[c] = first edge of the merged list whose node ends with a base >= c (A25): the node's last base is the first key
// symbol, so it is a lower bound over the solid edges plus one over the `$` nodes. One thread per c.
template <int W, int WT>
__global__ void edge_F_kernel(FullArgs a) {
    const u64 c = threadIdx.x;
    u64 lo = 0, hi = a.n;
    while (lo < hi) {
        const u64 mid = lo + ((hi - lo) >> 1);
        if ((a.keys[mid * W] >> 62) < c) lo = mid + 1; else hi = mid;
    }
    u64 lo2 = 0, hi2 = a.n_zero_out;
    while (lo2 < hi2) {
        const u64 mid = lo2 + ((hi2 - lo2) >> 1);
        if ((a.tk[(u64)a.zout_idx[mid] * WT] >> 62) < c) lo2 = mid + 1; else hi2 = mid;
    }
    a.F_dev[c] = lo + lo2;
}

// auxiliary vector: node i = src of edge zin_idx[i], bases in sequence order v[0..k), 2 bits each, node i at stream
// bits [2k i, 2k (i+1)), stream bit 0 = most significant bit of word 0 (aux_bits zeroed before)
template <int W>
__global__ void __launch_bounds__(256) aux_pack_kernel(FullArgs a) {
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < a.t; i += (u64)gridDim.x * blockDim.x) {
        u64 e[W];
        ld_rec<W>(a.keys, a.zin_idx[i], e);
        for (u32 j = 0; j < a.k; ++j) {
            const u32 s = a.k - 1u - j;                  // key symbol s holds base v[k-1-s]
            const u64 sym = (e[s >> 5] >> (62u - 2u * (s & 31u))) & 3ull;
            const u64 off = 2ull * a.k * i + 2ull * j;
            if (sym) atomicOr(&a.aux_bits[off >> 6], sym << (62u - (u32)(off & 63ull)));
        }
    }
}

__global__ void __launch_bounds__(256) valid_fill_kernel(u64 *valid, u64 m) {
    const u64 words = (m + 63) / 64;
    for (u64 w = (u64)blockIdx.x * blockDim.x + threadIdx.x; w < words; w += (u64)gridDim.x * blockDim.x)
        valid[w] = (w + 1 < words || (m & 63) == 0) ? ~0ull : (~0ull >> (64 - (m & 63)));
}

static unsigned grid_for(u64 n) {
    u64 b = (n + 255) / 256;
    if (b == 0) b = 1;
    const u64 cap = (u64)num_sms() * 16;
    return (unsigned)(b < cap ? b : cap);
}

// (W, WT) pairs that occur: WT = ceil(2k/64) is W or W-1
#define SDBG_DISPATCH_WWT(W_, WT_, CALL)                                             \
    switch ((W_) * 8 + (WT_)) {                                                      \
        case 1 * 8 + 1: { constexpr int W = 1, WT = 1; CALL; } break;                \
        case 2 * 8 + 1: { constexpr int W = 2, WT = 1; CALL; } break;                \
        case 2 * 8 + 2: { constexpr int W = 2, WT = 2; CALL; } break;                \
        case 3 * 8 + 2: { constexpr int W = 3, WT = 2; CALL; } break;                \
        case 3 * 8 + 3: { constexpr int W = 3, WT = 3; CALL; } break;                \
        case 4 * 8 + 3: { constexpr int W = 4, WT = 3; CALL; } break;                \
        case 4 * 8 + 4: { constexpr int W = 4, WT = 4; CALL; } break;                \
        default: return (int)cudaErrorInvalidValue;                                  \
    }

int launch_target_keys(const u64 *keys, u64 n, u32 k, u32 W_, u32 WT_, u64 *out, cudaStream_t s) {
    if (n == 0) return 0;
    SDBG_DISPATCH_WWT(W_, WT_, (target_keys_kernel<W, WT><<<grid_for(n), 256, 0, s>>>(keys, n, k, out)));
    return (int)cudaGetLastError();
}

u32 zero_flags_prefix_bits(u32 k) { return 2 * k < 20 ? 2 * k : 20; }
u64 zero_flags_index_bytes(u32 k) { return 2 * ((((1ull << zero_flags_prefix_bits(k)) + 1) * 4 + 255) / 256 * 256); }

int launch_zero_flags(const u64 *keys, u64 n, u32 k, u32 W_, u32 WT_, const u64 *tk_sorted, const u32 *last_real32,
                      u32 *prefix_index, uint8_t *flag_out, uint8_t *flag_in, cudaStream_t s) {
    if (n == 0) return 0;
    const u32 pb = zero_flags_prefix_bits(k);
    const u64 entries = (1ull << pb) + 1;
    u32 *idx_edges = prefix_index, *idx_tk = prefix_index + zero_flags_index_bytes(k) / 8;
    prefix_index_kernel<<<(unsigned)((entries + 255) / 256), 256, 0, s>>>(keys, n, W_, pb, idx_edges);
    prefix_index_kernel<<<(unsigned)((entries + 255) / 256), 256, 0, s>>>(tk_sorted, n, WT_, pb, idx_tk);
    SDBG_DISPATCH_WWT(W_, WT_, (flag_zero_out_kernel<W, WT><<<grid_for(n), 256, 0, s>>>(tk_sorted, n, keys, k, idx_edges, pb, flag_out),
                                flag_zero_in_kernel<W, WT><<<grid_for(n), 256, 0, s>>>(keys, n, last_real32, tk_sorted, k, idx_tk, pb, flag_in)));
    return (int)cudaGetLastError();
}

int launch_full_assemble(const FullArgs &a, u32 W_, u32 WT_, cudaStream_t s) {
    valid_fill_kernel<<<grid_for((a.n + a.n_zero_out + 63) / 64), 256, 0, s>>>(a.out_valid, a.n + a.n_zero_out);
    if (a.n == 0) return (int)cudaGetLastError();
    SDBG_DISPATCH_WWT(W_, WT_, (dummy_pos_kernel<W, WT><<<grid_for(a.n_zero_out), 256, 0, s>>>(a),
                                assemble_kernel<<<grid_for((a.n + a.n_zero_out + 63) / 4), 256, 0, s>>>(a),
                                aux_pack_kernel<W><<<grid_for(a.t), 256, 0, s>>>(a),
                                edge_F_kernel<W, WT><<<1, 4, 0, s>>>(a)));
    return (int)cudaGetLastError();
}

}  // namespace sdbg

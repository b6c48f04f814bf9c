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
// flag of a real edge: it has a node of its own and no outgoing base).
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

// flag_out[j] = tk[j] is the first of its value and no edge has it as its node; tk sorted
template <int W, int WT>
__global__ void __launch_bounds__(256) flag_zero_out_kernel(const u64 *__restrict__ tk, u64 n, const u64 *__restrict__ keys, u32 k,
                                                            uint8_t *__restrict__ flag) {
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
            u64 lo = 0, hi = n;                          // first edge whose node is not less than v
            while (lo < hi) {
                const u64 mid = lo + ((hi - lo) >> 1);
                u64 e[W];
                ld_rec<W>(keys, mid, e);
                if (node_cmp<W, WT>(e, v, k) < 0) lo = mid + 1; else hi = mid;
            }
            if (lo < n) {
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
                                                           const u64 *__restrict__ tk, u32 k, uint8_t *__restrict__ flag) {
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (u64)gridDim.x * blockDim.x) {
        bool z = false;
        if ((last_bits32[i >> 5] >> (i & 31)) & 1u) {
            u64 e[W];
            ld_rec<W>(keys, i, e);
            u64 lo = 0, hi = n;                          // first target that is not less than the node
            while (lo < hi) {
                const u64 mid = lo + ((hi - lo) >> 1);
                u64 v[WT];
                ld_rec<WT>(tk, mid, v);
                if (node_cmp<W, WT>(e, v, k) > 0) lo = mid + 1; else hi = mid;
            }
            z = true;
            if (lo < n) {
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
template <int W, int WT>
__global__ void __launch_bounds__(256) merge_real_kernel(FullArgs a) {
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += (u64)gridDim.x * blockDim.x) {
        u64 e[W];
        ld_rec<W>(a.keys, i, e);
        u64 lo = 0, hi = a.n_zero_out;                   // `$` edges whose node is less than mine come before me
        while (lo < hi) {
            const u64 mid = lo + ((hi - lo) >> 1);
            u64 v[WT];
            ld_rec<WT>(a.tk, a.zout_idx[mid], v);
            if (node_cmp<W, WT>(e, v, a.k) > 0) lo = mid + 1; else hi = mid;
        }
        const u64 pos = i + lo;
        a.out_W[pos] = a.W_real[i];
        a.out_mult[pos] = a.mult_in[i];
        if ((a.last_real32[i >> 5] >> (i & 31)) & 1u) atomicOr(&a.out_last32[pos >> 5], 1u << (pos & 31));
        if (a.out_zin32 && a.flag_in[i]) atomicOr(&a.out_zin32[pos >> 5], 1u << (pos & 31));
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

template <int W, int WT>
__global__ void __launch_bounds__(256) merge_dummy_kernel(FullArgs a) {
    for (u64 j = (u64)blockIdx.x * blockDim.x + threadIdx.x; j < a.n_zero_out; j += (u64)gridDim.x * blockDim.x) {
        u64 v[WT];
        ld_rec<WT>(a.tk, a.zout_idx[j], v);
        u64 lo = 0, hi = a.n;                            // real edges whose node is less than mine come before me
        while (lo < hi) {
            const u64 mid = lo + ((hi - lo) >> 1);
            u64 e[W];
            ld_rec<W>(a.keys, mid, e);
            if (node_cmp<W, WT>(e, v, a.k) < 0) lo = mid + 1; else hi = mid;
        }
        const u64 pos = j + lo;
        a.out_W[pos] = 0;                                // '$'
        a.out_mult[pos] = 0;
        atomicOr(&a.out_last32[pos >> 5], 1u << (pos & 31));   // the only edge of its node
    }
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
    const u64 cap = (u64)kNumSMs * 16;
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

int launch_zero_flags(const u64 *keys, u64 n, u32 k, u32 W_, u32 WT_, const u64 *tk_sorted, const u32 *last_real32,
                      uint8_t *flag_out, uint8_t *flag_in, cudaStream_t s) {
    if (n == 0) return 0;
    SDBG_DISPATCH_WWT(W_, WT_, (flag_zero_out_kernel<W, WT><<<grid_for(n), 256, 0, s>>>(tk_sorted, n, keys, k, flag_out),
                                flag_zero_in_kernel<W, WT><<<grid_for(n), 256, 0, s>>>(keys, n, last_real32, tk_sorted, k, flag_in)));
    return (int)cudaGetLastError();
}

int launch_full_assemble(const FullArgs &a, u32 W_, u32 WT_, cudaStream_t s) {
    valid_fill_kernel<<<grid_for((a.n + a.n_zero_out + 63) / 64), 256, 0, s>>>(a.out_valid, a.n + a.n_zero_out);
    if (a.n == 0) return (int)cudaGetLastError();
    SDBG_DISPATCH_WWT(W_, WT_, (merge_real_kernel<W, WT><<<grid_for(a.n), 256, 0, s>>>(a),
                                merge_dummy_kernel<W, WT><<<grid_for(a.n_zero_out), 256, 0, s>>>(a),
                                aux_pack_kernel<W><<<grid_for(a.t), 256, 0, s>>>(a),
                                edge_F_kernel<W, WT><<<1, 4, 0, s>>>(a)));
    return (int)cudaGetLastError();
}

}  // namespace sdbg

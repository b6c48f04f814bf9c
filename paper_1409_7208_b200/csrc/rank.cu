// rank.cu — rank/select over the arrays of the full graph and the two traversal maps built on them ("supports
// O(1) time traversal from a vertex to its neighbors"; Bowe et al.; readings A24-A26).
//
// Five bit-vectors over the m edges: B_c = (W is base c, minus flag clear) for c = A,C,G,T, and H = last & ~zin. Each is
// stored as 64-byte cells {u64 ones before the cell, 7 x 64 bits}: cell j covers edges [448 j, 448 j + 448), which are
// words 7j .. 7j+6 of a plain bit-vector, so a rank is ONE aligned 64-byte read (two sectors of one line) and a
// popcount of at most seven words. Select keeps, per vector, the cell of every 512-th one (a cell holds at most 448
// ones, so at most one sample falls into a cell), binary-searches the count words of the few cells between two samples
// and finishes inside the cell. A traversal query is a chain of three or four dependent random reads: the kernels are
// latency/sector bound, one thread per query, nothing staged.
#include "kernels.cuh"
#include <mutex>

namespace sdbg {

constexpr u32 kCellBits = 448, kCellWords = 8, kSelStep = 512;

__device__ __forceinline__ const u64 *cell_ptr(const IndexView &ix, int v, u64 cell) {
    return ix.cells + ((u64)v * ix.n_cells + cell) * kCellWords;
}

// ones of vector v at positions < x (x <= m)
__device__ __forceinline__ u64 rank_v(const IndexView &ix, int v, u64 x) {
    const u64 cell = x / kCellBits;
    const u32 off = (u32)(x - cell * kCellBits);
    const ulonglong2 *c2 = reinterpret_cast<const ulonglong2 *>(cell_ptr(ix, v, cell));
    const ulonglong2 a = c2[0], b = c2[1], c = c2[2], d = c2[3];
    const u64 w[7] = {a.y, b.x, b.y, c.x, c.y, d.x, d.y};
    u64 r = a.x;
#pragma unroll
    for (u32 q = 0; q < 7; ++q) {
        const int bits = (int)off - (int)(64 * q);
        if (bits >= 64) r += __popcll(w[q]);
        else if (bits > 0) r += __popcll(w[q] & (~0ull >> (64 - bits)));
    }
    return r;
}

// position of the r-th set bit of x (1 <= r <= popc(x)), LSB = position 0
__device__ __forceinline__ u32 select_in_word(u64 x, u32 r) {
    u32 pos = 0;
#pragma unroll
    for (u32 width = 32; width >= 1; width >>= 1) {
        const u32 c = __popcll(x & ((1ull << width) - 1ull));
        if (r > c) { r -= c; x >>= width; pos += width; }
    }
    return pos;
}

// position of the r-th one of vector v (1 <= r <= ones[v])
__device__ __forceinline__ u64 select_v(const IndexView &ix, int v, u64 r) {
    const u64 j = (r - 1) / kSelStep;
    u64 lo = ix.samples[v][j];
    u64 hi = (j + 1 < ix.n_samples[v]) ? ix.samples[v][j + 1] : ix.n_cells - 1;
    while (lo < hi) {                                    // last cell whose count word is below r
        const u64 mid = lo + ((hi - lo + 1) >> 1);
        if (cell_ptr(ix, v, mid)[0] < r) lo = mid; else hi = mid - 1;
    }
    const ulonglong2 *c2 = reinterpret_cast<const ulonglong2 *>(cell_ptr(ix, v, lo));
    const ulonglong2 a = c2[0], b = c2[1], c = c2[2], d = c2[3];
    const u64 w[7] = {a.y, b.x, b.y, c.x, c.y, d.x, d.y};
    u32 rem = (u32)(r - a.x);
    u32 q = 0;
    u64 word = w[0];
#pragma unroll
    for (u32 t = 0; t < 6; ++t) {
        const u32 pc = __popcll(w[t]);
        if (q == t && rem > pc) { rem -= pc; q = t + 1; word = w[t + 1]; }
    }
    return lo * kCellBits + 64ull * q + select_in_word(word, rem);
}

// ---- build ---------------------------------------------------------------------------------------------------------------
// 64 cells per block. Fill: one thread per 64-edge word (a warp reads 2 KiB of W in a row), seven words make a cell, so
// the 448 threads of a block fill exactly 64 cells; popcounts meet in shared memory, word 0 of a cell gets its count and
// the block its five sums. Then a one-block scan of the block sums, and a finish kernel that scans the 64 counts of a
// block in place and lets every cell that holds a (512 j + 1)-th one write its select sample.
constexpr u32 kIndexBlock = 64, kFillThreads = 7 * kIndexBlock;

__global__ void __launch_bounds__(kFillThreads) index_fill_kernel(const uint8_t *__restrict__ W, const u64 *__restrict__ last_bits,
                                                                  const u64 *__restrict__ zin_bits, u64 m, u64 n_cells, u64 *__restrict__ cells,
                                                                  u64 *__restrict__ block_sums /* [5][gridDim.x] */) {
    __shared__ uint8_t s_pc[5][kFillThreads];
    __shared__ u32 s_sum[5][kIndexBlock / 32];
    const u64 n_words = (m + 63) / 64;
    const u32 tid = threadIdx.x;
    const u64 wi = (u64)blockIdx.x * kFillThreads + tid, e0 = wi * 64;
    const u64 cell = (u64)blockIdx.x * kIndexBlock + tid / 7;
    u64 bits[5] = {0, 0, 0, 0, 0};
    if (e0 < m) {
        const u32 lim = (u32)(m - e0 < 64 ? m - e0 : 64);
        if (lim == 64) {
            const u64 *w8 = reinterpret_cast<const u64 *>(W + e0);           // e0 is a multiple of 64
#pragma unroll
            for (u32 g = 0; g < 8; ++g) {
                const u64 x = w8[g];
#pragma unroll
                for (u32 b = 0; b < 8; ++b) {
                    const u32 lab = (u32)(x >> (8 * b)) & 0xffu;
#pragma unroll
                    for (u32 c = 0; c < 4; ++c) bits[c] |= (u64)(lab == c + 1) << (8 * g + b);   // no dynamic index: registers
                }
            }
        } else {
            for (u32 b = 0; b < lim; ++b) {
                const u32 lab = W[e0 + b];
#pragma unroll
                for (u32 c = 0; c < 4; ++c) bits[c] |= (u64)(lab == c + 1) << b;
            }
        }
        if (wi < n_words) bits[4] = last_bits[wi] & ~zin_bits[wi];
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) {
        if (cell < n_cells) cells[((u64)v * n_cells + cell) * kCellWords + 1 + tid % 7] = bits[v];
        s_pc[v][tid] = (uint8_t)__popcll(bits[v]);
    }
    __syncthreads();
    if (tid < 5 * kIndexBlock) {                         // five groups of 64 threads: the counts of the 64 cells of vector v
        const u32 v = tid / kIndexBlock, lc = tid % kIndexBlock;
        u32 cnt = 0;
#pragma unroll
        for (u32 q = 0; q < 7; ++q) cnt += s_pc[v][7 * lc + q];
        const u64 c = (u64)blockIdx.x * kIndexBlock + lc;
        if (c < n_cells) cells[((u64)v * n_cells + c) * kCellWords] = cnt;
        u32 x = cnt;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        if ((tid & 31u) == 0) s_sum[v][(tid % kIndexBlock) >> 5] = x;
    }
    __syncthreads();
    if (tid < 5) {
        u64 t = 0;
        for (u32 w = 0; w < kIndexBlock / 32; ++w) t += s_sum[tid][w];
        block_sums[(u64)tid * gridDim.x + blockIdx.x] = t;
    }
}

// block v: exclusive scan of the block sums of vector v; totals[v] = ones of the vector
__global__ void __launch_bounds__(1024) index_scan_kernel(u64 *block_sums, u32 nblocks, u64 *totals) {
    __shared__ u64 s_w[32];
    __shared__ u64 s_carry;
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    u64 *base = block_sums + (u64)blockIdx.x * nblocks;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (u32 b0 = 0; b0 < nblocks; b0 += 1024) {
        const u32 i = b0 + tid;
        const u64 v = i < nblocks ? base[i] : 0ull;
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
        if (i < nblocks) base[i] = off + incl - v;
        __syncthreads();
        if (tid == 1023) s_carry = off + incl;
        __syncthreads();
    }
    if (tid == 0) totals[blockIdx.x] = s_carry;
}

// word 0 of every cell: count -> ones before the cell; samples[v][j] = cell of the (512 j + 1)-th one of vector v
__global__ void __launch_bounds__(kIndexBlock) index_finish_kernel(IndexView ix, const u64 *__restrict__ block_sums) {
    __shared__ u32 s_w[5][kIndexBlock / 32];
    const u32 lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const u64 cell = (u64)blockIdx.x * kIndexBlock + threadIdx.x;
    u64 *cells = const_cast<u64 *>(ix.cells);
    u32 cnt[5], incl[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) {
        cnt[v] = cell < ix.n_cells ? (u32)cells[((u64)v * ix.n_cells + cell) * kCellWords] : 0u;
        incl[v] = warp_incl_scan_add(cnt[v]);
        if (lane == 31) s_w[v][warp] = incl[v];
    }
    __syncthreads();
    if (cell >= ix.n_cells) return;
#pragma unroll
    for (int v = 0; v < 5; ++v) {
        u64 before = block_sums[(u64)v * gridDim.x + blockIdx.x] + incl[v] - cnt[v];
        for (u32 w = 0; w < warp; ++w) before += s_w[v][w];
        cells[((u64)v * ix.n_cells + cell) * kCellWords] = before;
        const u64 j = (before + kSelStep - 1) / kSelStep;        // smallest j with 512 j + 1 > before
        if (cnt[v] && j * kSelStep + 1 <= before + cnt[v]) ix.samples[v][j] = (u32)cell;
    }
}

// consts[c] = rank_H(F[c]) for c = 0..4
__global__ void index_consts_kernel(IndexView ix, u64 *consts) {
    const u32 c = threadIdx.x;
    if (c < 5) consts[c] = rank_v(ix, 4, ix.F[c]);
}

// ---- index build for callers that cannot allocate (sdbg_index_build_static) -----------------------------------------------
// The build scratch (16 scalars + five block sums per 64 cells) lives in a file-scope device array instead of the caller's
// block: 5 * ceil((2^28 / 448 + 1) / 64) + 16 words = 374,648 bytes, held by every GPU that loads the library until exit.
// Every call on a device shares it and it keeps the last call's contents: the scalars are cleared per call, the block sums
// are all overwritten before they are read. Calls that overlap on one GPU race on it.
constexpr u64 kStaticIndexMaxEdges = 1ull << 28;
constexpr u64 kStaticScratchWords = 5 * ((kStaticIndexMaxEdges / kCellBits + 1 + kIndexBlock - 1) / kIndexBlock) + 16;
static __device__ __align__(256) u64 g_index_scratch[kStaticScratchWords];

u64 index_static_max_edges() { return kStaticIndexMaxEdges; }

// Device address of g_index_scratch on the CURRENT device. In host code the array's name is a host-side stand-in, not a
// device address, so it is looked up once per device (with that device current) and kept.
static int index_static_scratch(u64 **ptr) {
    constexpr int kMaxDev = 64;
    static std::mutex mu;
    static u64 *cache[kMaxDev] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
    if (dev < 0 || dev >= kMaxDev) return (int)cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!cache[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_index_scratch);
        if (e != cudaSuccess) return (int)e;
        cache[dev] = static_cast<u64 *>(p);
    }
    *ptr = cache[dev];
    return 0;
}

// launch_index_build with the scratch above; *scratch_out = its device address (the scalars are read back from there)
int launch_index_build_static(const uint8_t *W, const u64 *last_bits, const u64 *zin_bits, const IndexView &ix, u64 **scratch_out, cudaStream_t s) {
    if (ix.m > kStaticIndexMaxEdges || index_scratch_words(ix.m) > kStaticScratchWords) return (int)cudaErrorInvalidValue;
    u64 *scratch = nullptr;
    int e = index_static_scratch(&scratch);
    if (e) return e;
    e = (int)cudaMemsetAsync(scratch, 0, 16 * sizeof(u64), s);
    if (e) return e;
    launch_index_build(W, last_bits, zin_bits, ix, scratch, s);
    *scratch_out = scratch;
    return (int)cudaGetLastError();
}

// ---- queries ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) forward_kernel(IndexView ix, const u64 *__restrict__ q, u64 n, long long *__restrict__ out) {
    for (u64 t = (u64)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (u64)gridDim.x * blockDim.x) {
        const u64 i = q[t];
        long long r = -2;
        if (i < ix.m) {
            const u32 lab = ix.W[i];
            r = -1;
            if (lab) {
                const u32 c = (lab - 1u) & 3u;
                r = (long long)select_v(ix, 4, ix.HF[c] + rank_v(ix, (int)c, i + 1));
            }
        }
        out[t] = r;
    }
}

__global__ void __launch_bounds__(256) backward_kernel(IndexView ix, const u64 *__restrict__ q, u64 n, long long *__restrict__ out) {
    for (u64 t = (u64)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (u64)gridDim.x * blockDim.x) {
        const u64 j = q[t];
        long long r = -2;
        if (j < ix.m) {
            u64 p = j;                                   // last edge of the node: at most four edges further on
            u64 word = ix.last_bits[p >> 6] >> (p & 63);
            if (word == 0) { p = (p | 63) + 1; word = ix.last_bits[p >> 6]; }
            p += __ffsll((long long)word) - 1;
            const u32 c = (p >= ix.F[1]) + (p >= ix.F[2]) + (p >= ix.F[3]);
            const u64 upto = rank_v(ix, 4, p + 1);
            const u64 before = rank_v(ix, 4, p);
            r = -1;
            if (upto != before) r = (long long)select_v(ix, (int)c, upto - ix.HF[c]);   // H[p] set: the node has an incoming edge
        }
        out[t] = r;
    }
}

static unsigned grid_q(u64 n) {
    u64 b = (n + 255) / 256;
    if (b == 0) b = 1;
    const u64 cap = (u64)num_sms() * 32;
    return (unsigned)(b < cap ? b : cap);
}

u64 index_cells(u64 m) { return m / kCellBits + 1; }
u64 index_samples_cap(u64 m) { return m / kSelStep + 2; }

u64 index_scratch_words(u64 m) { return 5 * ((index_cells(m) + kIndexBlock - 1) / kIndexBlock) + 16; }

// scratch: u64[index_scratch_words(m)]: 16 scalars (ones of the five vectors at [0..4], rank_H(F[c]) at [8..12]), block sums
void launch_index_build(const uint8_t *W, const u64 *last_bits, const u64 *zin_bits, const IndexView &ix, u64 *scratch, cudaStream_t s) {
    const u32 nblocks = (u32)((ix.n_cells + kIndexBlock - 1) / kIndexBlock);
    u64 *block_sums = scratch + 16;
    index_fill_kernel<<<nblocks, kFillThreads, 0, s>>>(W, last_bits, zin_bits, ix.m, ix.n_cells, const_cast<u64 *>(ix.cells), block_sums);
    index_scan_kernel<<<5, 1024, 0, s>>>(block_sums, nblocks, scratch);
    index_finish_kernel<<<nblocks, kIndexBlock, 0, s>>>(ix, block_sums);
    index_consts_kernel<<<1, 32, 0, s>>>(ix, scratch + 8);
}

void launch_forward(const IndexView &ix, const u64 *q, u64 n, long long *out, cudaStream_t s) {
    if (n) forward_kernel<<<grid_q(n), 256, 0, s>>>(ix, q, n, out);
}
void launch_backward(const IndexView &ix, const u64 *q, u64 n, long long *out, cudaStream_t s) {
    if (n) backward_kernel<<<grid_q(n), 256, 0, s>>>(ix, q, n, out);
}

}  // namespace sdbg

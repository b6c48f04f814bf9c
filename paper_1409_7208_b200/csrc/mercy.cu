// mercy.cu — mercy-kmers (§2 ¶3; readings A21-A23 of DESIGN.md): "Given two solid
// (k+1)-mers x and y from the same read, where x has no outdegree and y has no indegree. If all (k+1)-mers between x
// and y in that read are not solid, they will be added to the de Bruijn graph as mercy-kmers."
//
// Second scan of the packed reads. One thread per end mark of the `ends` bit-vector = per read: it walks the read's
// windows with a rolling key (the key of the next window is the target-node key of the current one with the new base
// appended), looks every window up in the sorted solid edges (binary search), and for every maximal run of non-solid
// windows with a solid window x before it and a solid window y behind it tests tgt(x) against the nodes without
// outgoing edge and src(y) against the nodes without incoming edge (the lists of sdbg_build_full). The windows of a
// qualifying run and their reverse complements are appended to the output (one atomicAdd per run).
#include "kernels.cuh"

namespace sdbg {

template <int W>
__device__ __forceinline__ void ldk(const u64 *__restrict__ a, u64 i, u64 (&k)[W]) {
#pragma unroll
    for (int q = 0; q < W; ++q) k[q] = a[i * W + q];
}
template <int W>
__device__ __forceinline__ int cmpk(const u64 (&a)[W], const u64 (&b)[W]) {
#pragma unroll
    for (int q = 0; q < W; ++q) if (a[q] != b[q]) return a[q] < b[q] ? -1 : 1;
    return 0;
}
// keep the top `bits` bits of a W-word value
template <int W>
__device__ __forceinline__ void mask_top(u64 (&v)[W], u32 bits) {
#pragma unroll
    for (int q = 0; q < W; ++q) {
        const int rem = (int)bits - 64 * q;
        v[q] &= rem >= 64 ? ~0ull : rem <= 0 ? 0ull : ~0ull << (64 - rem);
    }
}
__device__ __forceinline__ u64 base_at(const u64 *__restrict__ words, u64 slot) {
    return (__ldg(words + (slot >> 5)) >> (62u - 2u * (u32)(slot & 31))) & 3ull;
}
// symbol s (0 = most significant) of a W-word key
template <int W>
__device__ __forceinline__ void set_sym(u64 (&v)[W], u32 s, u64 sym) {
#pragma unroll
    for (int q = 0; q < W; ++q) if ((s >> 5) == (u32)q) v[q] |= sym << (62u - 2u * (s & 31u));
}

// forward key (e[k-1],...,e[0],e[k]) and rc-strand key (c(e[1]),...,c(e[k]),c(e[0])) of the window starting at `slot`
template <int W>
__device__ void window_keys(const u64 *__restrict__ words, u64 slot, u32 k, u64 (&f)[W], u64 (&r)[W]) {
#pragma unroll
    for (int q = 0; q < W; ++q) { f[q] = 0; r[q] = 0; }
    for (u32 j = 0; j <= k; ++j) {
        const u64 b = base_at(words, slot + j);
        set_sym<W>(f, j < k ? k - 1u - j : k, b);            // e[j] sits at symbol k-1-j; e[k] at symbol k
        set_sym<W>(r, j == 0 ? k : j - 1u, 3ull - b);        // c(e[j]) sits at symbol j-1; c(e[0]) at symbol k
    }
}

// Hash table over the solid edges (open addressing, linear probing, load <= 1/2). A slot is 16 bytes: the first key word
// and edge index + 1 (0 = empty), so a look-up of a one-word key is ONE random 16-byte read (the key is compared in the
// slot itself); longer keys compare their first word there and the remaining words through the index only when it
// matches. The build claims a slot with a CAS on the index field and then stores the key word: nothing reads the table
// before the build kernel has ended, and the edges are distinct, so no key is compared while building.
template <int W>
__device__ __forceinline__ u64 hash_key(const u64 (&key)[W]) {
    u64 h = 0;
#pragma unroll
    for (int q = 0; q < W; ++q) h = mix64(h ^ key[q]);
    return h;
}
template <int W>
__global__ void __launch_bounds__(256) hash_build_kernel(const u64 *__restrict__ keys, u64 n, ulonglong2 *__restrict__ table, u64 mask) {
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (u64)gridDim.x * blockDim.x) {
        u64 key[W];
        ldk<W>(keys, i, key);
        u64 h = hash_key<W>(key) & mask;
        while (atomicCAS(reinterpret_cast<u32 *>(&table[h].y), 0u, (u32)i + 1u) != 0u) h = (h + 1) & mask;
        table[h].x = key[0];
    }
}
void launch_hash_build(const u64 *keys, u64 n, u32 W, void *table, u64 slots, cudaStream_t s) {
    u64 blocks = (n + 255) / 256;
    if (blocks > (u64)num_sms() * 16) blocks = (u64)num_sms() * 16;
    if (blocks == 0) return;
    ulonglong2 *t = reinterpret_cast<ulonglong2 *>(table);
    switch (W) {
        case 1: hash_build_kernel<1><<<(unsigned)blocks, 256, 0, s>>>(keys, n, t, slots - 1); break;
        case 2: hash_build_kernel<2><<<(unsigned)blocks, 256, 0, s>>>(keys, n, t, slots - 1); break;
        case 3: hash_build_kernel<3><<<(unsigned)blocks, 256, 0, s>>>(keys, n, t, slots - 1); break;
        default: hash_build_kernel<4><<<(unsigned)blocks, 256, 0, s>>>(keys, n, t, slots - 1); break;
    }
}

template <int W>
__device__ __forceinline__ bool is_solid(const MercyArgs &a, const u64 (&key)[W]) {
    const ulonglong2 *table = reinterpret_cast<const ulonglong2 *>(a.table);
    u64 h = hash_key<W>(key) & a.table_mask;
    while (true) {
        const ulonglong2 v = __ldg(table + h);
        const u32 idx1 = (u32)v.y;
        if (idx1 == 0u) return false;
        if (v.x == key[0]) {
            bool same = true;
#pragma unroll
            for (int q = 1; q < W; ++q) same = same && __ldg(a.keys + ((u64)idx1 - 1u) * W + q) == key[q];
            if (same) return true;
        }
        h = (h + 1) & a.table_mask;
    }
}

// node (top 2k bits of `key`, W words) among the nodes without outgoing edge (tk rows listed by zout_idx, WT words)
template <int W, int WT>
__device__ __forceinline__ bool in_zero_out(const MercyArgs &a, const u64 (&node)[W]) {
    u64 lo = 0, hi = a.n_zero_out;
    while (lo < hi) {
        const u64 mid = lo + ((hi - lo) >> 1);
        u64 v[WT];
        ldk<WT>(a.tk, a.zout_idx[mid], v);
        int c = 0;
#pragma unroll
        for (int q = 0; q < WT; ++q) if (c == 0 && v[q] != node[q]) c = v[q] < node[q] ? -1 : 1;
        if (c == 0) return true;
        if (c < 0) lo = mid + 1; else hi = mid;
    }
    return false;
}
template <int W>
__device__ __forceinline__ bool in_zero_in(const MercyArgs &a, const u64 (&node)[W]) {
    u64 lo = 0, hi = a.t;
    while (lo < hi) {
        const u64 mid = lo + ((hi - lo) >> 1);
        u64 e[W];
        ldk<W>(a.keys, a.zin_idx[mid], e);
        mask_top<W>(e, 2 * a.k);
        const int c = cmpk<W>(e, node);
        if (c == 0) return true;
        if (c < 0) lo = mid + 1; else hi = mid;
    }
    return false;
}

template <int W, int WT>
__global__ void __launch_bounds__(128) mercy_kernel(MercyArgs a, DevState *st) {
    const u32 k = a.k, pad = 64u * W - 2u * (k + 1u);
    const u64 nwords = a.n_slots / 64;
    for (u64 wi = (u64)blockIdx.x * blockDim.x + threadIdx.x; wi < nwords; wi += (u64)gridDim.x * blockDim.x) {
        u64 marks = __ldg(a.ends + wi);
        while (marks) {
            const u32 bit = (u32)__ffsll((long long)marks) - 1u;
            marks &= marks - 1;
            const u64 last = wi * 64 + bit;                      // last base slot of a read (or a padding slot)
            // first slot of the read: the slot after the previous end mark
            u64 first = 0;
            {
                u64 m = bit ? (__ldg(a.ends + wi) & ((1ull << bit) - 1ull)) : 0ull;
                long long w2 = (long long)wi;
                while (m == 0 && w2 > 0) { --w2; m = __ldg(a.ends + w2); }
                if (m) first = (u64)w2 * 64 + (63u - (u32)__clzll((long long)m)) + 1;
            }
            const u64 L = last - first + 1;
            if (L < (u64)k + 3) continue;                        // fewer than 3 windows: no run can have both neighbours
            const u64 nw = L - k;
            u64 key[W], prev[W], unused[W];
            window_keys<W>(a.words, first, k, key, unused);
            bool prev_solid = false, left_ok = false;
            long long run_start = -1;
            for (u64 i = 0; i < nw; ++i) {
                if (i) {   // rolling key: target-node key of the previous window, then the new outgoing base
                    const u64 last_sym = (key[W - 1] >> pad) & 3ull;
#pragma unroll
                    for (int q = W - 1; q >= 0; --q) key[q] = (key[q] >> 2) | (q ? key[q - 1] << 62 : 0ull);
                    key[0] |= last_sym << 62;
                    mask_top<W>(key, 2 * k);
                    set_sym<W>(key, k, base_at(a.words, first + i + k));
                }
                const bool sol = is_solid<W>(a, key);
                if (!sol) {
                    if (run_start < 0) {
                        run_start = (long long)i;
                        left_ok = false;
                        if (i > 0 && prev_solid) {               // x = window i-1: tgt(x) = node part of my key
                            u64 node[W];
#pragma unroll
                            for (int q = 0; q < W; ++q) node[q] = key[q];
                            mask_top<W>(node, 2 * k);
                            left_ok = in_zero_out<W, WT>(a, node);
                        }
                    }
                } else {
                    if (run_start >= 0 && left_ok) {             // y = this window: src(y) = its node
                        u64 node[W];
#pragma unroll
                        for (int q = 0; q < W; ++q) node[q] = key[q];
                        mask_top<W>(node, 2 * k);
                        if (in_zero_in<W>(a, node)) {
                            const u64 cnt = 2 * (i - (u64)run_start);
                            const u64 base = atomicAdd(&st->extract_cursor, cnt);
                            if (base + cnt <= a.out_cap) {
                                u64 f[W], r[W];
                                window_keys<W>(a.words, first + (u64)run_start, k, f, r);
                                for (u64 j = (u64)run_start; j < i; ++j) {
                                    if (j > (u64)run_start) {    // both keys roll on by the base that enters the window
                                        const u64 nb = base_at(a.words, first + j + k);
                                        const u64 f_last = (f[W - 1] >> pad) & 3ull, r_first = r[0] >> 62;
#pragma unroll
                                        for (int q = W - 1; q >= 0; --q) f[q] = (f[q] >> 2) | (q ? f[q - 1] << 62 : 0ull);
                                        f[0] |= f_last << 62;
                                        mask_top<W>(f, 2 * k);
                                        set_sym<W>(f, k, nb);
#pragma unroll
                                        for (int q = 0; q < W; ++q) r[q] = (r[q] << 2) | (q + 1 < W ? r[q + 1] >> 62 : 0ull);
                                        mask_top<W>(r, 2 * (k - 1));
                                        set_sym<W>(r, k - 1, 3ull - nb);
                                        set_sym<W>(r, k, r_first);
                                    }
                                    const u64 o = base + 2 * (j - (u64)run_start);
#pragma unroll
                                    for (int q = 0; q < W; ++q) { a.out_keys[o * W + q] = f[q]; a.out_keys[(o + 1) * W + q] = r[q]; }
                                    a.out_mult[o] = 1; a.out_mult[o + 1] = 1;
                                }
                            }
                        }
                    }
                    run_start = -1;
                }
                prev_solid = sol;
                (void)prev;
            }
        }
    }
}

int launch_mercy(const MercyArgs &a, u32 W_, u32 WT_, DevState *st, cudaStream_t s) {
    const u64 nwords = a.n_slots / 64;
    if (nwords == 0 || a.n == 0) return 0;
    u64 blocks = (nwords + 127) / 128;
    if (blocks > (u64)num_sms() * 32) blocks = (u64)num_sms() * 32;
    const unsigned g = (unsigned)blocks;
    switch (W_ * 8 + WT_) {
        case 1 * 8 + 1: mercy_kernel<1, 1><<<g, 128, 0, s>>>(a, st); break;
        case 2 * 8 + 1: mercy_kernel<2, 1><<<g, 128, 0, s>>>(a, st); break;
        case 2 * 8 + 2: mercy_kernel<2, 2><<<g, 128, 0, s>>>(a, st); break;
        case 3 * 8 + 2: mercy_kernel<3, 2><<<g, 128, 0, s>>>(a, st); break;
        case 3 * 8 + 3: mercy_kernel<3, 3><<<g, 128, 0, s>>>(a, st); break;
        case 4 * 8 + 3: mercy_kernel<4, 3><<<g, 128, 0, s>>>(a, st); break;
        case 4 * 8 + 4: mercy_kernel<4, 4><<<g, 128, 0, s>>>(a, st); break;
        default: return (int)cudaErrorInvalidValue;
    }
    return (int)cudaGetLastError();
}

}  // namespace sdbg

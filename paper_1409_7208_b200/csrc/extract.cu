// extract.cu — step a2: every (k+1)-window of the packed reads -> two sort keys (forward edge and
// its reverse complement; "all (k+1)-mers from the input reads", both strands per reading A4/A5),
// with the digit histograms of all LSD passes and the 65,536-bin l=8 partition histogram fused in.
//
// Key of edge e = symbols (e[k-1],...,e[0],e[k]) MSB-first (include/sdbg.h). For the window e at slot p:
//   forward key : reversed node ++ e[k]          = rot(Y),  Y = (e[k], e[k-1], ..., e[0]) taken from the
//                                                  2-bit-group-reversed word stream;
//   rc key      : (c(e[1]),...,c(e[k]),c(e[0]))  = rot(~win), win = (e[0],...,e[k]) taken from the forward stream;
// where rot moves the first symbol of a (k+1)-symbol string to its end (identity checked in the tests against
// the string oracle). One thread owns 32 consecutive slots, one warp 1024; keys leave the warp in coalesced
// runs at a position reserved with one atomicAdd per warp (the order of raw records is irrelevant: they are sorted).
#include "kernels.cuh"

namespace sdbg {

// shared-memory atomics by 32-bit shared address (one LEA in front of the ATOMS / RED instead of the address arithmetic
// of a generic pointer); the hot loops below issue two to four of them per window
__device__ __forceinline__ u32 smem_addr(const void *p) { return (u32)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void s_inc(u32 addr) { asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(addr) : "memory"); }
__device__ __forceinline__ void s_add(u32 addr, u32 v) { asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory"); }
__device__ __forceinline__ u32 s_fetch_inc(u32 addr) {
    u32 r;
    asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(r) : "r"(addr) : "memory");
    return r;
}
__device__ __forceinline__ void s_st64(u32 addr, u64 v) { asm volatile("st.shared.u64 [%0], %1;" ::"r"(addr), "l"(v) : "memory"); }

__device__ __forceinline__ u64 rev2(u64 x) {   // reverse the order of the 32 2-bit groups
    u32 lo = (u32)x, hi = (u32)(x >> 32);
    u64 y = ((u64)__brev(lo) << 32) | (u64)__brev(hi);
    return ((y >> 1) & 0x5555555555555555ull) | ((y & 0x5555555555555555ull) << 1);
}
// top 64 bits of the 128-bit value (hi:lo) << s, s in [0, 63]
__device__ __forceinline__ u64 funnel(u64 hi, u64 lo, u32 s) { return s ? ((hi << s) | (lo >> (64 - s))) : hi; }

template <int W>
struct KeyMaker {
    u64 B[W + 1];    // forward stream: slots 32g .. 32g+32(W+1)
    u64 R[W + 1];    // reversed stream, pre-shifted so that Y_i starts at symbol 31-i
    u32 k;
    u64 lastmask;

    __device__ __forceinline__ void load(const u64 *__restrict__ words, u64 g, u32 k_) {
        k = k_;
        lastmask = ~0ull << (64 * W - 2 * (k + 1));
#pragma unroll
        for (int j = 0; j <= W; ++j) B[j] = __ldg(words + g + j);
        u64 T[W + 2];
#pragma unroll
        for (int j = 0; j <= W; ++j) T[j] = rev2(B[W - j]);
        T[W + 1] = 0;
        const u32 q0 = 32 * (W + 1) - k - 32;   // 1..32 symbols
        if (q0 == 32) {
#pragma unroll
            for (int j = 0; j <= W; ++j) R[j] = T[j + 1];
        } else {
#pragma unroll
            for (int j = 0; j <= W; ++j) R[j] = funnel(T[j], T[j + 1], 2 * q0);
        }
    }
    // rot: first symbol of the (k+1)-symbol string to its end
    __device__ __forceinline__ void rot(const u64 (&V)[W], u64 (&out)[W]) const {
        const u64 top = V[0] >> 62;
#pragma unroll
        for (int j = 0; j < W; ++j) out[j] = (V[j] << 2) | (j + 1 < W ? (V[j + 1] >> 62) : 0ull);
        out[W - 1] |= top << (62 - 2 * (k & 31));
    }
    // The same for window i = 16 HALF + ii with 32-bit funnel shifts: the word pairs are fixed by HALF, only the
    // shift amount (< 32) is a run-time value, so a 64-bit window costs two SHF instead of a dozen instructions.
    template <int HALF>
    __device__ __forceinline__ void keys_h(u32 ii, u64 (&fwd)[W], u64 (&rc)[W]) const {
        u64 win[W], Y[W];
        const u32 s = 2 * ii, t = 30 - 2 * ii;    // bit offsets 32 HALF + s (forward) and 32 (1 - HALF) + t (reversed)
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const u32 wh = __funnelshift_l(w32(B, 2 * j + HALF + 1), w32(B, 2 * j + HALF), s);
            const u32 wl = __funnelshift_l(w32(B, 2 * j + HALF + 2), w32(B, 2 * j + HALF + 1), s);
            const u32 yh = __funnelshift_l(w32(R, 2 * j + 2 - HALF), w32(R, 2 * j + 1 - HALF), t);
            const u32 yl = __funnelshift_l(w32(R, 2 * j + 3 - HALF), w32(R, 2 * j + 2 - HALF), t);
            win[j] = ~(((u64)wh << 32) | wl);
            Y[j] = ((u64)yh << 32) | yl;
        }
        win[W - 1] &= lastmask;
        Y[W - 1] &= lastmask;
        rot(Y, fwd);
        rot(win, rc);
    }
    // l=8 partitions (top 16 key bits) of both keys of window i = 16 HALF + ii, for k >= 8: symbols 1..8 of the
    // reversed-stream window (forward key) and of the complemented forward window (rc-strand key); two funnel shifts
    template <int HALF>
    __device__ __forceinline__ void buckets_h(u32 ii, u32 &bf, u32 &br) const {
        const u32 wh = __funnelshift_l(w32(B, HALF + 1), w32(B, HALF), 2 * ii);
        const u32 yh = __funnelshift_l(w32(R, 2 - HALF), w32(R, 1 - HALF), 30 - 2 * ii);
        bf = (yh >> 14) & 0xffffu;
        br = (~wh >> 14) & 0xffffu;
    }
    // 32-bit word m of a stream of u64 words, most significant first
    static __device__ __forceinline__ u32 w32(const u64 (&S)[W + 1], int m) { return (m & 1) ? (u32)S[m >> 1] : (u32)(S[m >> 1] >> 32); }
    __device__ __forceinline__ void keys(u32 i, u64 (&fwd)[W], u64 (&rc)[W]) const {
        u64 win[W], Y[W];
        const u32 s = 2 * i, t = 2 * (31 - i);
#pragma unroll
        for (int j = 0; j < W; ++j) {
            win[j] = ~funnel(B[j], B[j + 1], s);
            Y[j] = funnel(R[j], R[j + 1], t);
        }
        win[W - 1] &= lastmask;
        Y[W - 1] &= lastmask;
        rot(Y, fwd);
        rot(win, rc);
    }
};

template <int W>
__device__ __forceinline__ void store_key(u64 *__restrict__ out, u64 pos, const u64 (&key)[W]) {
    if constexpr (W == 1) {
        out[pos] = key[0];
    } else if constexpr (W == 2) {
        *reinterpret_cast<ulonglong2 *>(out + pos * 2) = make_ulonglong2(key[0], key[1]);
    } else if constexpr (W == 4) {
        *reinterpret_cast<ulonglong2 *>(out + pos * 4) = make_ulonglong2(key[0], key[1]);
        *reinterpret_cast<ulonglong2 *>(out + pos * 4 + 2) = make_ulonglong2(key[2], key[3]);
    } else {
#pragma unroll
        for (int j = 0; j < W; ++j) out[pos * W + j] = key[j];
    }
}

constexpr int kCoarseBins = 4096;   // groups of 16 consecutive l=8 partitions (ExtractArgs::coarse_hist)

template <int W, bool FILTER, int T4>
__global__ void __launch_bounds__(256) extract_kernel(ExtractArgs a, DevState *st) {
    extern __shared__ u32 s_hist[];   // [n_passes][256] when digit_hist != nullptr
    const int np = a.passes.n;
    const bool do_hist = a.digit_hist != nullptr;
    // T4 >= 2 (one-word keys, dense pass, digit histograms wanted, T4 = floor(k/4)): the T4 top key bytes hold node symbols
    // only, and byte t of the forward key of the window at slot p is the reversed 4-mer at x = p + k-4-4t, byte t of the
    // rc-strand key the complemented 4-mer at x = p + 4t + 1. So a read position x contributes the SAME byte value to
    // the histograms of a contiguous range of t (all T4 of them in the interior of a read, fewer near its ends: the
    // window starts that exist are an interval). Positions are therefore counted as differences over t — +1 in row
    // t_lo, -1 in row t_hi + 1 — in two position tables indexed by the plain 4-mer f4 (forward strand: its symbol
    // reversal is the digit; rc strand: its complement), prefix-summed over t and folded into the pass rows when the
    // block flushes. For k >= 8 exactly one key byte is left (byte 7 - T4 from the LSB, the one with e[k]): it is the
    // only per-key atomic. Shared-memory atomics, the bottleneck of this kernel, drop from 8 per key to about 2.4.
    constexpr bool shared4 = T4 >= 2;
    constexpr u32 T = shared4 ? T4 : 0;
    u32 *s_posf = s_hist + np * kRadix, *s_posr = s_posf + (T + 1) * kRadix;   // [T + 1][256] each (shared4 only); row T is a spare
    if (do_hist) {
        for (int i = threadIdx.x; i < (np + (shared4 ? 2 * (int)T + 2 : 0)) * kRadix; i += blockDim.x) s_hist[i] = 0;
        __syncthreads();
    } else if (a.coarse_hist) {
        for (int i = threadIdx.x; i < kCoarseBins; i += blockDim.x) s_hist[i] = 0;
        __syncthreads();
    }
    // s_hist row of byte 0 of the last key word if it were a pass (rows of the padding bytes are never touched)
    const u32 b0 = a.passes.n ? (u32)a.passes.p[0].shift >> 3 : 0u;
    // one-word keys, a.hist_top most significant passes wanted only: bytes below bmin of the key word are not counted
    const u32 bmin = (W == 1 && a.hist_top && (int)a.hist_top < np) ? b0 + (u32)np - a.hist_top : b0;
    // the same for any key width, without position tables: rows of word 0 start at h_word0 (indexed by the byte of the word),
    // its bytes top_lo .. 7 are wanted
    const bool top_only = !shared4 && a.hist_top != 0 && a.hist_top <= 4u && (W > 1 || (int)a.hist_top < np);
    const u32 top_lo = W == 1 ? bmin : 8u - a.hist_top;
    const u32 hist_s = smem_addr(s_hist);
    const u32 h_word0_s = hist_s + 4u * (u32)(W == 1 ? 0 : ((8 - b0) + 8 * (W - 2)) * kRadix) - (W == 1 ? 4u * b0 * kRadix : 0u);
    const u32 posf_s = hist_s + 4u * (u32)(np * kRadix), posr_s = posf_s + 4u * (T + 1) * kRadix;
    const u64 ngroups = a.n_slots / 32;
    const u32 lane = lane_id();
    const u32 lt = lanemask_lt();
    u64 csum = 0;

    // warp-granular grid-stride loop: warp handles groups [32*wg, 32*wg+32)
    const u64 nwarp_groups = (ngroups + 31) / 32;
    const u64 warps_total = (u64)gridDim.x * (blockDim.x >> 5);
    for (u64 wg = (u64)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); wg < nwarp_groups; wg += warps_total) {
        const u64 g = wg * 32 + lane;
        u32 valid = (g < ngroups) ? valid_mask32(a.ends, g, a.k) : 0u;
        u32 vprev = 0;                                   // valid window starts of the 32 slots before mine
        if constexpr (shared4) {
            vprev = __shfl_up_sync(0xffffffffu, valid, 1);
            if (lane == 0) vprev = (g >= 1 && g - 1 < ngroups) ? valid_mask32(a.ends, g - 1, a.k) : 0u;
        }
        if (__ballot_sync(0xffffffffu, (valid | vprev) != 0) == 0) continue;
        KeyMaker<W> km;
        km.load(a.words, g < ngroups ? g : 0, a.k);
        if constexpr (!FILTER && !shared4) {
            if (a.coarse_hist) {   // planner's histogram: top 12 key bits of both keys of every window, shared-memory counters
#pragma unroll 4
                for (u32 ii = 0; ii < 16; ++ii) {
                    u32 bf, br;
                    km.template buckets_h<0>(ii, bf, br);
                    if ((valid >> ii) & 1u) { s_inc(hist_s + 4u * (bf >> 4)); s_inc(hist_s + 4u * (br >> 4)); }
                }
#pragma unroll 4
                for (u32 ii = 0; ii < 16; ++ii) {
                    u32 bf, br;
                    km.template buckets_h<1>(ii, bf, br);
                    if ((valid >> (16 + ii)) & 1u) { s_inc(hist_s + 4u * (bf >> 4)); s_inc(hist_s + 4u * (br >> 4)); }
                }
                continue;
            }
        }
        if constexpr (shared4) {
            if (valid | vprev) {
                // window starts [32g-32, 32g+32) as one mask: bit 32+j = start at my slot j
                const u64 V = ((u64)valid << 32) | vprev;
                constexpr u32 pat = 0x11111111u >> (4 * (8 - T));       // bits 0, 4, ..., 4(T-1)
                const u32 off_f = 32 - (a.k - 4), off_r = 32 - 1 - 4 * (T - 1);
                auto count_pos = [&](u32 j, u32 f4) {   // f4 = (r[x], r[x+1], r[x+2], r[x+3]) at my slot j
                    const u32 mf = (u32)(V >> (off_f + j)) & pat;       // bit 4t: the window whose forward byte t I am
                    const u32 mr = (u32)(V >> (off_r + j)) & pat;       // bit 4(T-1-t): the window whose rc byte t I am
                    // branch-free: a position without window (mask 0) and a range that ends at T go to the spare row T
                    const u32 f_lo = ((u32)__ffs(mf) - 1u) >> 2, f_end = ((31u - (u32)__clz(mf)) >> 2) + 1u;
                    s_inc(posf_s + 4u * ((mf ? f_lo : T) * kRadix + f4));
                    s_add(posf_s + 4u * ((mf ? f_end : T) * kRadix + f4), 0xffffffffu);
                    const u32 r_lo = T - 1u - ((31u - (u32)__clz(mr)) >> 2), r_end = T - (((u32)__ffs(mr) - 1u) >> 2);
                    s_inc(posr_s + 4u * ((mr ? r_lo : T) * kRadix + f4));
                    s_add(posr_s + 4u * ((mr ? r_end : T) * kRadix + f4), 0xffffffffu);
                };
                const u32 b0w = KeyMaker<W>::w32(km.B, 0), b1w = KeyMaker<W>::w32(km.B, 1), b2w = KeyMaker<W>::w32(km.B, 2);
#pragma unroll 4
                for (u32 jj = 0; jj < 16; ++jj) count_pos(jj, __funnelshift_l(b1w, b0w, 2 * jj) >> 24);
#pragma unroll 4
                for (u32 jj = 0; jj < 16; ++jj) count_pos(16 + jj, __funnelshift_l(b2w, b1w, 2 * jj) >> 24);
            }
        }
        if constexpr (shared4) {
            // histogram-only call for the top passes (the pre-scan of the fused extract-and-scatter path): the position
            // tables hold everything that is wanted, no key is made
            if (!a.keys_out && !a.bucket_hist && !a.want_csum && bmin > 7u - T) continue;
        }
        u32 vf = valid, vr = valid;   // per-strand keep masks
        if (FILTER && a.k >= 8) {
            // which keys fall into the range of partitions: only the top 16 bits of each key are needed
            const u32 lo = a.bucket_lo, span = a.bucket_hi - a.bucket_lo;
            u32 mf = 0, mr = 0;
#pragma unroll 4
            for (u32 ii = 0; ii < 16; ++ii) {
                u32 bf, br;
                km.template buckets_h<0>(ii, bf, br);
                mf |= (u32)(bf - lo < span) << ii;
                mr |= (u32)(br - lo < span) << ii;
            }
#pragma unroll 4
            for (u32 ii = 0; ii < 16; ++ii) {
                u32 bf, br;
                km.template buckets_h<1>(ii, bf, br);
                mf |= (u32)(bf - lo < span) << (16 + ii);
                mr |= (u32)(br - lo < span) << (16 + ii);
            }
            vf = mf & valid; vr = mr & valid;
        } else if (FILTER) {
            vf = 0; vr = 0;
            for (u32 i = 0; i < 32; ++i) {
                if (!((valid >> i) & 1)) continue;
                u64 f[W], r[W];
                km.keys(i, f, r);
                u32 bf = (u32)(f[0] >> 48), br = (u32)(r[0] >> 48);
                if (bf >= a.bucket_lo && bf < a.bucket_hi) vf |= 1u << i;
                if (br >= a.bucket_lo && br < a.bucket_hi) vr |= 1u << i;
            }
        }
        u64 base = 0;
        if (a.keys_out) {
            u32 cnt = __popc(vf) + __popc(vr);
            u32 incl = warp_incl_scan_add(cnt);
            u32 total = __shfl_sync(0xffffffffu, incl, 31);
            if (lane == 0 && total) base = atomicAdd(&st->extract_cursor, (u64)total);
            base = __shfl_sync(0xffffffffu, base, 0);
            if (base + total > a.out_cap) continue;   // cannot happen when the caller sized out_cap from the histogram
        }
        // digit histograms of one key: every pass is one whole byte of a key word (api.cu make_passes): byte b of word
        // q is pass (b - b0) for the last word and (8 - b0) + 8 (W-2-q) + b for the others, b0 = first significant byte
        auto add_digits = [&](const u64 (&key)[W]) {
            if constexpr (shared4) {   // the one byte that is not counted by position: byte 7 - T from the LSB = pass 0
                constexpr u32 b = 7 - T;
                if (bmin <= b) s_inc(hist_s + 4u * __byte_perm(b < 4 ? (u32)key[0] : (u32)(key[0] >> 32), 0u, 0x4440u | (b & 3)));
            } else if (top_only) {
                // rows of the hist_top most significant passes only: the top bytes of word 0, a short loop without predicates
                const u32 hi = (u32)(key[0] >> 32);                  // at most four top passes (api_count.inc plan_hash)
#pragma unroll
                for (u32 b = 7; b >= 4; --b)
                    if (b >= top_lo) s_inc(h_word0_s + 4u * (b * kRadix + __byte_perm(hi, 0u, 0x4440u | (b & 3u))));
            } else {
#pragma unroll
                for (int q = W - 1; q >= 0; --q) {
                    if (W > 1 && q > 0 && a.hist_top) continue;      // (keys of several words) top passes only: bytes of word 0
                    const u32 hq_s = (q == W - 1) ? hist_s - 4u * b0 * kRadix : hist_s + 4u * (u32)(((8 - b0) + 8 * (W - 2 - q)) * kRadix);
                    const u32 lo = (u32)key[q], hi = (u32)(key[q] >> 32);
#pragma unroll
                    for (int b = 0; b < 8; ++b) {
                        if (q == W - 1 && b < (int)bmin) continue;   // padding bytes of the last word (and passes not wanted): no row
                        if (W > 1 && a.hist_top && b + (int)a.hist_top < 8) continue;
                        s_inc(hq_s + 4u * (b * kRadix + __byte_perm(b < 4 ? lo : hi, 0u, 0x4440u | (b & 3))));
                    }
                }
            }
        };
        // (keys of several words, table-count path) the one-word stand-in of the record at output place pos, and its index
        auto put_pair = [&](u64 pos, const u64 (&key)[W]) {
            a.pair_keys[pos] = pair_key<W>(key, a.pair_top_bits & 0xffu, (a.pair_top_bits >> 8) != 0);
            a.pair_idx[pos] = (u32)pos;
        };
        // one key per lane (or none): coalesced store at the warp's running position, digit histograms, checksum
        auto emit_key = [&](bool keep, const u64 (&key)[W]) {
            if (a.keys_out) {
                const u32 m = __ballot_sync(0xffffffffu, keep);
                if (keep) {
                    store_key<W>(a.keys_out, base + __popc(m & lt), key);
                    if constexpr (W > 1) if (a.pair_keys) put_pair(base + __popc(m & lt), key);
                }
                base += __popc(m);
            }
            if (keep) {
                if (do_hist) add_digits(key);
                if (a.want_csum) csum += mix_key<W>(key);
            }
        };
        if (FILTER && a.k >= 8) {
            // block-wise pass: a lane keeps only a few of its 64 keys, so it walks over the set bits of its keep masks
            // (its own window index per step) instead of over all 32 windows
            u32 rem_f = vf, rem_r = vr;
            while (__any_sync(0xffffffffu, (rem_f | rem_r) != 0)) {
                const bool hf = rem_f != 0, hr = rem_r != 0;
                const u32 i_f = hf ? (u32)__ffs(rem_f) - 1u : 0u, i_r = hr ? (u32)__ffs(rem_r) - 1u : 0u;
                rem_f &= rem_f - 1u;
                rem_r &= rem_r - 1u;
                u64 f[W], r[W], unused[W];
                km.keys(i_f, f, unused);
                km.keys(i_r, unused, r);
                emit_key(hf, f);
                emit_key(hr, r);
            }
        } else {
            const u32 any_mask = __reduce_or_sync(0xffffffffu, valid);
            auto emit_window = [&](u32 i, const u64 (&f)[W], const u64 (&r)[W]) {
                const bool kf = (vf >> i) & 1, kr = (vr >> i) & 1;
                if (a.keys_out) {
                    const u32 mf = __ballot_sync(0xffffffffu, kf), mr = __ballot_sync(0xffffffffu, kr);
                    if (kf) {
                        store_key<W>(a.keys_out, base + __popc(mf & lt), f);
                        if constexpr (W > 1) if (a.pair_keys) put_pair(base + __popc(mf & lt), f);
                    }
                    base += __popc(mf);
                    if (kr) {
                        store_key<W>(a.keys_out, base + __popc(mr & lt), r);
                        if constexpr (W > 1) if (a.pair_keys) put_pair(base + __popc(mr & lt), r);
                    }
                    base += __popc(mr);
                }
                if (do_hist) {
                    if (kf) add_digits(f);
                    if (kr) add_digits(r);
                }
                if (a.want_csum) {
                    if (kf) csum += mix_key<W>(f);
                    if (kr) csum += mix_key<W>(r);
                }
                if (a.bucket_hist && ((valid >> i) & 1)) {
                    atomicAdd(&a.bucket_hist[f[0] >> 48], 1ull);
                    atomicAdd(&a.bucket_hist[r[0] >> 48], 1ull);
                }
            };
            // the plain case of the hot path (one-word keys, keys and digit histograms wanted, no checksum, no partition
            // histogram): both keys of a window leave as ONE 16-byte store under one predicate (the warp's running
            // position stays even: every lane adds two keys per window)
            bool fast = false;
            if constexpr (W == 1) fast = a.keys_out && do_hist && !a.want_csum && !a.bucket_hist;
            auto emit_fast = [&](u32 i, const u64 (&f)[W], const u64 (&r)[W]) {
                const bool v = (valid >> i) & 1;
                const u32 m = __ballot_sync(0xffffffffu, v);
                if (v) {
                    *reinterpret_cast<ulonglong2 *>(a.keys_out + base + 2 * __popc(m & lt)) = make_ulonglong2(f[0], r[0]);
                    add_digits(f);
                    add_digits(r);
                }
                base += 2 * __popc(m);
            };
            if (fast) {
#pragma unroll 1
                for (u32 ii = 0; ii < 16; ++ii) {
                    if (!((any_mask >> ii) & 1)) continue;     // warp-uniform
                    u64 f[W], r[W];
                    km.template keys_h<0>(ii, f, r);
                    emit_fast(ii, f, r);
                }
#pragma unroll 1
                for (u32 ii = 0; ii < 16; ++ii) {
                    if (!((any_mask >> (16 + ii)) & 1)) continue;
                    u64 f[W], r[W];
                    km.template keys_h<1>(ii, f, r);
                    emit_fast(16 + ii, f, r);
                }
            } else {
#pragma unroll 1
                for (u32 ii = 0; ii < 16; ++ii) {
                    if (!((any_mask >> ii) & 1)) continue;     // warp-uniform
                    u64 f[W], r[W];
                    km.template keys_h<0>(ii, f, r);
                    emit_window(ii, f, r);
                }
#pragma unroll 1
                for (u32 ii = 0; ii < 16; ++ii) {
                    if (!((any_mask >> (16 + ii)) & 1)) continue;
                    u64 f[W], r[W];
                    km.template keys_h<1>(ii, f, r);
                    emit_window(16 + ii, f, r);
                }
            }
        }
    }
    if (a.want_csum) {
        csum = warp_reduce_add64(csum);
        if (lane == 0 && csum) atomicAdd(&st->csum_raw, csum);
    }
    if (!do_hist && a.coarse_hist) {
        __syncthreads();
        for (int i = threadIdx.x; i < kCoarseBins; i += blockDim.x) {
            const u32 v = s_hist[i];
            if (v) atomicAdd(&a.coarse_hist[i], (u64)v);
        }
    }
    if (do_hist) {
        __syncthreads();
        if constexpr (shared4) {
            // position tables: differences over t -> counts (prefix sums, top byte first) ...
            for (u32 dgt = threadIdx.x; dgt < (u32)kRadix; dgt += blockDim.x) {
                u32 rf = 0, rr = 0;
                for (u32 t = 0; t < T; ++t) {
                    rf += s_posf[t * kRadix + dgt]; s_posf[t * kRadix + dgt] = rf;
                    rr += s_posr[t * kRadix + dgt]; s_posr[t * kRadix + dgt] = rr;
                }
            }
            __syncthreads();
            // ... folded into the pass rows: byte t is pass T - t; digit d of the forward strand is the symbol reversal of
            // f4, of the rc strand its complement
            for (u32 i = threadIdx.x; i < T * (u32)kRadix; i += blockDim.x) {
                const u32 t = i >> kRadixBits, dgt = i & (kRadix - 1);
                const u32 rev = ((dgt & 0x03u) << 6) | ((dgt & 0x0cu) << 2) | ((dgt & 0x30u) >> 2) | ((dgt & 0xc0u) >> 6);
                s_hist[(T - t) * kRadix + dgt] = s_posf[t * kRadix + rev] + s_posr[t * kRadix + (~dgt & 0xffu)];
            }
            __syncthreads();
        }
        for (int i = threadIdx.x; i < np * kRadix; i += blockDim.x) {
            u32 v = s_hist[i];
            if (v) atomicAdd(&a.digit_hist[i], (u64)v);
        }
    }
}

// ---- keys of several words, table-count path, few valid windows per slot (ExtractArgs::by_rows) --------------------------------
// A warp takes one group of 32 base slots per step, lane = slot. The valid-window mask of the group is the same for all
// lanes, so a group without a window costs one mask; in a group with windows every lane that has one makes both keys (the
// KeyMaker of the group, window = lane), and the records, their one-word stand-ins and indices leave the warp together.
// Digit rows of the hist_top top passes only (the caller's table-count path), no filter, no checksum.
template <int W>
__global__ void __launch_bounds__(256) extract_rows_kernel(ExtractArgs a, DevState *st) {
    extern __shared__ u32 s_hist[];   // [n_passes][256]; only the rows of the top passes of word 0 are touched
    const int np = a.passes.n;
    for (int i = threadIdx.x; i < np * kRadix; i += blockDim.x) s_hist[i] = 0;
    __syncthreads();
    const u32 b0 = a.passes.n ? (u32)a.passes.p[0].shift >> 3 : 0u;
    const u32 top_lo = 8u - a.hist_top;
    const u32 h_word0_s = smem_addr(s_hist) + 4u * (u32)(((8 - b0) + 8 * (W - 2)) * kRadix);
    const u64 ngroups = a.n_slots / 32;
    const u32 lane = lane_id(), lt = lanemask_lt();
    const u32 top_bits = a.pair_top_bits & 0xffu;
    const bool weak = (a.pair_top_bits >> 8) != 0;
    const u64 warps_total = (u64)gridDim.x * (blockDim.x >> 5);
    const u64 nspans = (ngroups + 31) / 32;              // a warp takes 32 consecutive groups at a time: one reservation of output
    for (u64 sp = (u64)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); sp < nspans; sp += warps_total) {
        const u64 g0 = sp * 32;
        const u32 my_valid = g0 + lane < ngroups ? valid_mask32(a.ends, g0 + lane, a.k) : 0u;   // lane j: the mask of group g0 + j
        const u32 total = 2u * (u32)__reduce_add_sync(0xffffffffu, (u32)__popc(my_valid));
        if (total == 0) continue;
        u64 base = 0;
        if (lane == 0) base = atomicAdd(&st->extract_cursor, (u64)total);
        base = __shfl_sync(0xffffffffu, base, 0);
        if (base + total > a.out_cap) continue;          // cannot happen when the caller sized out_cap from the window count
        u32 groups = __ballot_sync(0xffffffffu, my_valid != 0);
        while (groups) {
            const u32 j = (u32)__ffs(groups) - 1u;
            groups &= groups - 1u;
            const u32 valid = __shfl_sync(0xffffffffu, my_valid, j);
            KeyMaker<W> km;
            km.load(a.words, g0 + j, a.k);
            u64 f[W], r[W];
            km.keys(lane, f, r);
            const bool v = (valid >> lane) & 1u;
            if (v) {
                const u64 pos = base + 2 * __popc(valid & lt);
                store_key<W>(a.keys_out, pos, f);
                store_key<W>(a.keys_out, pos + 1, r);
                if (a.pair_keys) {
                    a.pair_keys[pos] = pair_key<W>(f, top_bits, weak);
                    a.pair_keys[pos + 1] = pair_key<W>(r, top_bits, weak);
                    *reinterpret_cast<uint2 *>(a.pair_idx + pos) = make_uint2((u32)pos, (u32)pos + 1u);   // pos is even
                }
                const u32 fh = (u32)(f[0] >> 32), rh = (u32)(r[0] >> 32);
#pragma unroll
                for (u32 b = 7; b >= 4; --b) {
                    if (b >= top_lo) {
                        s_inc(h_word0_s + 4u * (b * kRadix + __byte_perm(fh, 0u, 0x4440u | (b & 3u))));
                        s_inc(h_word0_s + 4u * (b * kRadix + __byte_perm(rh, 0u, 0x4440u | (b & 3u))));
                    }
                }
            }
            base += 2 * __popc(valid);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < np * kRadix; i += blockDim.x) {
        const u32 c = s_hist[i];
        if (c) atomicAdd(&a.digit_hist[i], (u64)c);
    }
}

// ---- extraction fused with the first (unstable) radix pass --------------------------------------------------------------
// One-word keys, dense range, default path (api_count.inc): the keys are not written in read order and re-read by the
// first top pass; they go straight from the key maker into the 256 bins of that pass. The bin sizes come from a
// histogram-only pre-scan of the packed reads (extract_kernel without output: position tables, 0.375 bytes per base).
// The digit is key byte `t` from the top (t < floor(k / 4): a byte of node symbols only), so that for the window at slot p
//   forward key: digit = symbol reversal of the 4-mer at slot p + k - 4 - 4t,   rc-strand key: complement of the 4-mer at
//   slot p + 4t + 1  (the identity extract_kernel's position tables use).
// Per tile of 4,096 slots (8 warps x 32 lanes x 16 slots; a lane owns half a group of 32 slots):
//   A  digits of all valid windows counted by the plain 4-mer in two 256-entry tables (no key is made), folded into the
//      tile's bin counts (reversal / complement of the index);
//   B  one thread per bin: exclusive scan -> tile place of the bin; its run in the output is reserved with ONE atomicAdd
//      on the bin's global cursor (the order of the records inside a bin is free: they are merged or sorted later);
//   C  the keys are made, each takes the next place of its bin in shared memory (shared atomic), 
//   D  and the tile leaves in bin order: place p goes to (reserved run of its bin) + (p - tile place of the bin), one
//      coalesced run per bin.
struct ScatterSmem {
    static constexpr int THREADS = 256, TILE_GROUPS = 128, MAX_KEYS = TILE_GROUPS * 32 * 2;
    static constexpr size_t kStage = 0;                                   // u64[MAX_KEYS]
    static constexpr size_t kCntF = kStage + (size_t)MAX_KEYS * 8;        // u32[256] digits of forward keys by plain 4-mer
    static constexpr size_t kCntR = kCntF + 1024;                         // u32[256] digits of rc-strand keys by plain 4-mer
    static constexpr size_t kCur = kCntR + 1024;                          // u32[256] next free tile place of the bin
    static constexpr size_t kOff = kCur + 1024;                           // u64[256] output index of tile place 0 if it were in this bin
    static constexpr size_t kBytes = kOff + 2048;
};

template <int HALF>
__device__ __forceinline__ void scatter_count_half(const KeyMaker<1> &km, u32 valid16, u64 S0f, u64 S1f, u64 S0r, u64 S1r,
                                                   u32 cntF_s, u32 cntR_s) {   // 32-bit shared addresses of the two tables
#pragma unroll
    for (u32 ii = 0; ii < 16; ++ii) {
        constexpr u32 base = 16u * HALF;
        const u32 j = base + ii;                          // window = slot j of the group; its 4-mers start at symbol j of S
        const u32 f4 = j <= 28 ? (u32)(S0f >> (56 - 2 * j)) & 0xffu : (u32)(funnel(S0f, S1f, 2 * j) >> 56);
        const u32 r4 = j <= 28 ? (u32)(S0r >> (56 - 2 * j)) & 0xffu : (u32)(funnel(S0r, S1r, 2 * j) >> 56);
        if ((valid16 >> ii) & 1u) { s_inc(cntF_s + 4u * f4); s_inc(cntR_s + 4u * r4); }
    }
}

template <int HALF>
__device__ __forceinline__ void scatter_place_half(const KeyMaker<1> &km, u32 valid16, u32 dshift, u32 cur_s, u32 stage_s) {
#pragma unroll
    for (u32 ii = 0; ii < 16; ++ii) {
        u64 f[1], r[1];
        km.template keys_h<HALF>(ii, f, r);
        if ((valid16 >> ii) & 1u) {
            const u32 pf = s_fetch_inc(cur_s + 4u * ((u32)(f[0] >> dshift) & 0xffu));
            const u32 pr = s_fetch_inc(cur_s + 4u * ((u32)(r[0] >> dshift) & 0xffu));
            s_st64(stage_s + 8u * pf, f[0]);
            s_st64(stage_s + 8u * pr, r[0]);
        }
    }
}

__global__ void __launch_bounds__(ScatterSmem::THREADS, 3) extract_scatter_kernel(ScatterArgs a) {
    using L = ScatterSmem;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    u64 *s_stage = reinterpret_cast<u64 *>(smem_raw + L::kStage);
    u32 *s_cntF = reinterpret_cast<u32 *>(smem_raw + L::kCntF), *s_cntR = reinterpret_cast<u32 *>(smem_raw + L::kCntR);
    u32 *s_cur = reinterpret_cast<u32 *>(smem_raw + L::kCur);
    u64 *s_off = reinterpret_cast<u64 *>(smem_raw + L::kOff);
    const u32 smem_s = smem_addr(smem_raw);
    const u32 stage_s = smem_s + (u32)L::kStage, cntF_s = smem_s + (u32)L::kCntF, cntR_s = smem_s + (u32)L::kCntR, cur_s = smem_s + (u32)L::kCur;
    __shared__ u32 s_wtot[8];
    __shared__ u32 s_total;
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const u32 half = warp >> 2;                          // warps 0-3: slots 0-15 of their groups, warps 4-7: slots 16-31
    const u64 ngroups = a.n_slots / 32;
    const u64 ntiles = (ngroups + L::TILE_GROUPS - 1) / L::TILE_GROUPS;
    const u32 off_f = a.k - 4u - 4u * a.t, off_r = 4u * a.t + 1u, dshift = 56u - 8u * a.t;
    s_cntF[tid] = 0; s_cntR[tid] = 0;
    __syncthreads();
    for (u64 tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const u64 g = tile * L::TILE_GROUPS + 32u * (warp & 3u) + lane;
        u32 valid16 = 0;
        KeyMaker<1> km;
        if (g < ngroups) valid16 = (valid_mask32(a.ends, g, a.k) >> (16u * half)) & 0xffffu;
        const bool any = __any_sync(0xffffffffu, valid16 != 0);
        if (any) km.load(a.words, g < ngroups ? g : 0, a.k);
        // ---- A: digits by plain 4-mer
        if (valid16) {
            const u64 S0f = funnel(km.B[0], km.B[1], 2 * off_f), S1f = off_f ? km.B[1] << (2 * off_f) : km.B[1];
            const u64 S0r = funnel(km.B[0], km.B[1], 2 * off_r), S1r = km.B[1] << (2 * off_r);
            if (half) scatter_count_half<1>(km, valid16, S0f, S1f, S0r, S1r, cntF_s, cntR_s);
            else scatter_count_half<0>(km, valid16, S0f, S1f, S0r, S1r, cntF_s, cntR_s);
        }
        __syncthreads();
        // ---- B: bin tid: count (fold), exclusive scan over the bins, reservation of its run in the output
        {
            const u32 rev = ((tid & 0x03u) << 6) | ((tid & 0x0cu) << 2) | ((tid & 0x30u) >> 2) | ((tid & 0xc0u) >> 6);
            const u32 c = s_cntF[rev] + s_cntR[~tid & 0xffu];
            const u32 incl = warp_incl_scan_add(c);
            if (lane == 31) s_wtot[warp] = incl;
            __syncthreads();
            u32 start = incl - c;
            for (u32 w = 0; w < warp; ++w) start += s_wtot[w];
            s_cur[tid] = start;
            u64 gpos = 0;
            if (c) gpos = atomicAdd(&a.bin_cursor[tid], (u64)c);
            s_off[tid] = gpos - start;
            if (tid == 255) s_total = start + c;
            __syncthreads();
            s_cntF[tid] = 0; s_cntR[tid] = 0;            // for the next tile (their readers are past the barrier above)
        }
        // ---- C: keys into their bins in shared memory
        if (valid16) {
            if (half) scatter_place_half<1>(km, valid16, dshift, cur_s, stage_s);
            else scatter_place_half<0>(km, valid16, dshift, cur_s, stage_s);
        }
        __syncthreads();
        // ---- D: the tile leaves in bin order
        const u32 total = s_total;
        for (u32 p = tid; p < total; p += L::THREADS) {
            const u64 key = s_stage[p];
            const u64 dst = s_off[(u32)(key >> dshift) & 0xffu] + p;
            if (dst < a.out_cap) a.keys_out[dst] = key;
        }
        __syncthreads();
    }
}

int extract_scatter_setup() {
    return (int)cudaFuncSetAttribute(extract_scatter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ScatterSmem::kBytes);
}

bool extract_scatter_supported(u32 k, u32 t) { return k >= 8 && k <= 31 && t < k / 4; }

int launch_extract_scatter(const ScatterArgs &a, cudaStream_t s) {
    const u64 ngroups = a.n_slots / 32;
    if (ngroups == 0) return 0;
    if (!extract_scatter_supported(a.k, a.t)) return (int)cudaErrorInvalidValue;
    const u64 ntiles = (ngroups + ScatterSmem::TILE_GROUPS - 1) / ScatterSmem::TILE_GROUPS;
    const u64 cap = (u64)num_sms() * 3;
    extract_scatter_kernel<<<(unsigned)(ntiles < cap ? ntiles : cap), ScatterSmem::THREADS, ScatterSmem::kBytes, s>>>(a);
    return (int)cudaGetLastError();
}

template <int W>
static int launch_extract_w(const ExtractArgs &a, DevState *st, cudaStream_t s) {
    const u64 ngroups = a.n_slots / 32;
    if (ngroups == 0) return 0;
    const bool filter = !(a.bucket_lo == 0 && a.bucket_hi >= 65536);
    u64 blocks = (ngroups + 255) / 256;
    const u64 maxb = (u64)num_sms() * 8;
    if (blocks > maxb) blocks = maxb;
    const u32 T = (W == 1 && !filter && a.digit_hist && a.k >= 8) ? a.k / 4 : 0;   // 2..7: shared position tables
    size_t smem = a.digit_hist ? (size_t)(a.passes.n + (T ? 2 * T + 2 : 0)) * kRadix * sizeof(u32) : 0;
    if (a.coarse_hist) {   // histogram-only call of the planner
        if (a.digit_hist || a.bucket_hist || a.keys_out || a.want_csum || filter || a.k < 8) return (int)cudaErrorInvalidValue;
        smem = (size_t)kCoarseBins * sizeof(u32);
    }
    if (filter) { extract_kernel<W, true, 0><<<(unsigned)blocks, 256, smem, s>>>(a, st); return (int)cudaGetLastError(); }
    if constexpr (W > 1) {
        if (a.by_rows) {
            if (!a.keys_out || !a.digit_hist || !a.hist_top || a.hist_top > 4 || a.want_csum || a.bucket_hist || a.coarse_hist)
                return (int)cudaErrorInvalidValue;
            extract_rows_kernel<W><<<(unsigned)maxb, 256, smem, s>>>(a, st);
            return (int)cudaGetLastError();
        }
    }
    if constexpr (W == 1) {
        switch (T) {
            case 2: extract_kernel<1, false, 2><<<(unsigned)blocks, 256, smem, s>>>(a, st); return (int)cudaGetLastError();
            case 3: extract_kernel<1, false, 3><<<(unsigned)blocks, 256, smem, s>>>(a, st); return (int)cudaGetLastError();
            case 4: extract_kernel<1, false, 4><<<(unsigned)blocks, 256, smem, s>>>(a, st); return (int)cudaGetLastError();
            case 5: extract_kernel<1, false, 5><<<(unsigned)blocks, 256, smem, s>>>(a, st); return (int)cudaGetLastError();
            case 6: extract_kernel<1, false, 6><<<(unsigned)blocks, 256, smem, s>>>(a, st); return (int)cudaGetLastError();
            case 7: extract_kernel<1, false, 7><<<(unsigned)blocks, 256, smem, s>>>(a, st); return (int)cudaGetLastError();
            default: break;
        }
    }
    extract_kernel<W, false, 0><<<(unsigned)blocks, 256, smem, s>>>(a, st);
    return (int)cudaGetLastError();
}

int launch_extract(const ExtractArgs &a, DevState *st, cudaStream_t s) {
    switch (a.W) {
        case 1: return launch_extract_w<1>(a, st, s);
        case 2: return launch_extract_w<2>(a, st, s);
        case 3: return launch_extract_w<3>(a, st, s);
        case 4: return launch_extract_w<4>(a, st, s);
    }
    return (int)cudaErrorInvalidValue;
}

}  // namespace sdbg

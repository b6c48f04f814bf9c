// emit.cu — step a5: the BOSS-style SdBG arrays from the sorted solid edges (§2 ¶1,
// Bowe et al. 2012 PAPER.md:106; flag rules per BASELINE.json north_star, readings A10, A14):
//   W[i]     = e[k]                                  (byte 1..4 = A,C,G,T; +4 when minus; 0 reserved for '$')
//   last[i]  = (i == n-1) or node(i+1) != node(i)    node = the k symbols before the last one of the key
//   minus[i] = exists j < i with e_j[1..k) == e_i[1..k) and e_j[k] == e_i[k]
// In key order (e[k-1],...,e[1],e[0],e[k]) the edges sharing e[1..k) share the top 2(k-1) key bits, so they are
// contiguous (at most 16 of them: 4 values of e[0] x 4 of e[k]) and the scan over j stops after at most 15 steps.
#include "kernels.cuh"

namespace sdbg {

// true iff the top `nbits` bits of the W-word keys a and b are equal (nbits in [0, 64W])
template <int W>
__device__ __forceinline__ bool top_bits_equal(const u64 (&a)[W], const u64 (&b)[W], u32 nbits) {
    bool eq = true;
#pragma unroll
    for (int q = 0; q < W; ++q) {
        const u32 lo = 64u * q;
        if (nbits > lo) {
            const u32 nb = nbits - lo >= 64u ? 64u : nbits - lo;            // bits of this word that take part
            const u64 mask = nb == 64u ? ~0ull : ~(~0ull >> nb);
            eq = eq && (((a[q] ^ b[q]) & mask) == 0);
        }
    }
    return eq;
}

template <int W>
__device__ __forceinline__ void ld_key(const u64 *__restrict__ keys, u64 i, u64 (&k)[W]) {
#pragma unroll
    for (int q = 0; q < W; ++q) k[q] = __ldg(keys + i * W + q);
}

template <int W>
__global__ void __launch_bounds__(256) emit_kernel(EmitArgs a) {
    const u32 lane = lane_id();
    const u32 k = a.k;
    const u32 wsh = 64u * W - 2u * (k + 1u);          // bit offset of the last symbol in the last word
    const u64 nround = (a.n + 31) / 32 * 32;          // whole warps so that the ballot covers the tail
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < nround; i += (u64)gridDim.x * blockDim.x) {
        bool last = false;
        if (i < a.n) {
            u64 me[W];
            ld_key<W>(a.keys, i, me);
            const u32 wsym = (u32)(me[W - 1] >> wsh) & 3u;
            last = true;
            if (i + 1 < a.n) {
                u64 nx[W];
                ld_key<W>(a.keys, i + 1, nx);
                last = !top_bits_equal<W>(me, nx, 2u * k);
            }
            bool minus = false;
            for (u64 j = i; j-- > 0;) {
                u64 pk[W];
                ld_key<W>(a.keys, j, pk);
                if (!top_bits_equal<W>(me, pk, 2u * (k - 1u))) break;
                if (((u32)(pk[W - 1] >> wsh) & 3u) == wsym) { minus = true; break; }
            }
            a.Wout[i] = (uint8_t)(1u + wsym + (minus ? 4u : 0u));
            a.mult_out[i] = a.mult_in[i];
        }
        const u32 bits = __ballot_sync(0xffffffffu, last);
        if (lane == 0) a.last_bits32[i >> 5] = bits;
    }
}

void launch_emit(const EmitArgs &a, cudaStream_t s) {
    if (a.n == 0) return;
    u64 blocks = (a.n + 255) / 256;
    if (blocks > (u64)num_sms() * 16) blocks = (u64)num_sms() * 16;
    switch (a.W) {
        case 1: emit_kernel<1><<<(unsigned)blocks, 256, 0, s>>>(a); break;
        case 2: emit_kernel<2><<<(unsigned)blocks, 256, 0, s>>>(a); break;
        case 3: emit_kernel<3><<<(unsigned)blocks, 256, 0, s>>>(a); break;
        case 4: emit_kernel<4><<<(unsigned)blocks, 256, 0, s>>>(a); break;
    }
}

}  // namespace sdbg

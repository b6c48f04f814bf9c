// pack.cu — step a1: ASCII reads -> 2-bit packed reads + read-end marks, and the window counter.
//
// Packed layout (private to the library; see include/sdbg.h sdbg_reads):
//   words[i]  : base slots 32i..32i+31, slot p in bits [63-2(p%32) : 62-2(p%32)] (first base in the top bits),
//               A=0 C=1 G=2 T=3 (reading A1).
//   ends[i]   : bit (p%64) of ends[p/64] = 1 iff slot p is the last base of a read or a padding/guard slot.
// A (k+1)-window starting at slot p is a record iff no end mark lies in [p, p+k): then p..p+k are k+1 bases of
// one read ("(k+1)-mers from the input reads"; reads shorter than k+1 give none, reading A6).
#include "kernels.cuh"

namespace sdbg {

// 4 ASCII bytes (little-endian in x) -> 8 bits of codes, first byte in the top 2 bits; ok=false on non-ACGT.
__device__ __forceinline__ u32 pack4(u32 x, bool &ok) {
    u32 f = x & 0xDFDFDFDFu;                               // fold case
    u32 c = ((f >> 1) ^ (f >> 2)) & 0x03030303u;           // A0 C1 G2 T3 per byte
    // expected letters from the codes: 'A' + {0,2,6,19}
    u32 is1 = c & 0x01010101u, is2 = (c >> 1) & 0x01010101u;
    // letter = 0x41 + 2*is1 + 6*is2 + 11*(is1&is2)
    u32 both = is1 & is2;
    u32 expect = 0x41414141u + 2u * is1 + 6u * is2 + 11u * both;
    ok = ok && (expect == f);
    u32 b0 = c & 3u, b1 = (c >> 8) & 3u, b2 = (c >> 16) & 3u, b3 = (c >> 24) & 3u;
    return (b0 << 6) | (b1 << 4) | (b2 << 2) | b3;
}

// One thread per output word (32 bases). `ascii` points at the first base of the chunk, which maps to slot0
// (slot0 % 64 == 0). Bases beyond nb are written as 0 (they carry end marks).
__global__ void __launch_bounds__(256) pack_kernel(const unsigned char *__restrict__ ascii, u64 nb, u64 *__restrict__ words,
                                                   u64 slot0, u64 err_index_base, DevState *st) {
    const u64 nwords = (nb + 31) / 32;
    for (u64 j = (u64)blockIdx.x * blockDim.x + threadIdx.x; j < nwords; j += (u64)gridDim.x * blockDim.x) {
        const u64 a0 = j * 32;
        u64 word = 0;
        bool ok = true;
        if (a0 + 32 <= nb && ((reinterpret_cast<uintptr_t>(ascii + a0) & 15) == 0)) {
            const uint4 *p = reinterpret_cast<const uint4 *>(ascii + a0);
            uint4 v0 = __ldg(p), v1 = __ldg(p + 1);
            u32 q[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
#pragma unroll
            for (int t = 0; t < 8; ++t) word = (word << 8) | pack4(q[t], ok);
        } else {
            for (int t = 0; t < 32; ++t) {
                u32 ch = (a0 + t < nb) ? ascii[a0 + t] : 'A';
                bool o1 = true;
                u32 c = pack4(ch | 0x41414100u, o1) >> 6;
                ok = ok && o1;
                word = (word << 2) | c;
            }
        }
        if (!ok) {   // locate the first offending byte (rare path)
            u64 bad = ~0ull;
            for (int t = 31; t >= 0; --t) {
                if (a0 + t >= nb) continue;
                u32 f = ascii[a0 + t] & 0xDFu;
                if (f != 'A' && f != 'C' && f != 'G' && f != 'T') bad = err_index_base + a0 + t;
            }
            atomicMin(&st->bad_base, bad);
        }
        words[slot0 / 32 + j] = word;
    }
}

// One thread per read: set the end mark of its last base. Thread 0 also marks the padding slots of the chunk's
// final 64-group (pad_nb = bases of the call when this launch covers its first reads, else 0). `ends` words of the
// chunk were zeroed before. Every offset is bounded HERE, before it addresses anything: a read must satisfy
// off0 <= b <= e <= off0 + nb_total (non-decreasing offsets inside the span of the call); any other read is skipped
// and raises the flag (st->n_windows = ~0) that sdbg_pack_reads turns into SDBG_E_INVAL — a malformed offsets array
// never causes a write outside the chunk.
__global__ void __launch_bounds__(256) mark_ends_kernel(const u64 *__restrict__ offsets, u64 n, u64 off0, u64 nb_total, u64 pad_nb,
                                                        u64 *__restrict__ ends, u64 slot0, DevState *st) {
    u64 r = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (r == 0 && (pad_nb & 63)) atomicOr(&ends[(slot0 + pad_nb) >> 6], ~0ull << (pad_nb & 63));
    for (; r < n; r += (u64)gridDim.x * blockDim.x) {
        const u64 b = offsets[r], e = offsets[r + 1];
        if (b < off0 || e < b || e - off0 > nb_total) { st->n_windows = ~0ull; continue; }
        if (e > b) {
            const u64 p = slot0 + (e - 1 - off0);
            atomicOr(&ends[p >> 6], 1ull << (p & 63));
        }
    }
}

// Counts the valid (k+1)-windows: 32 slots per thread.
__global__ void __launch_bounds__(256) count_windows_kernel(const u64 *__restrict__ ends, u64 n_slots, u32 k, DevState *st) {
    u64 local = 0;
    const u64 ngroups = n_slots / 32;
    for (u64 g = (u64)blockIdx.x * blockDim.x + threadIdx.x; g < ngroups; g += (u64)gridDim.x * blockDim.x)
        local += __popc(valid_mask32(ends, g, k));
    local = warp_reduce_add64(local);
    if (lane_id() == 0 && local) atomicAdd(&st->n_windows, local);
}

void launch_pack(const unsigned char *d_ascii, u64 nb, u64 *words, u64 slot0, u64 err_index_base, DevState *st, cudaStream_t s) {
    if (nb == 0) return;
    u64 nwords = (nb + 31) / 32;
    u64 blocks = (nwords + 255) / 256;
    if (blocks > (u64)num_sms() * 16) blocks = (u64)num_sms() * 16;
    pack_kernel<<<(unsigned)blocks, 256, 0, s>>>(d_ascii, nb, words, slot0, err_index_base, st);
}

void launch_mark_ends(const u64 *d_offsets, u64 n, u64 off0, u64 nb_total, u64 pad_nb, u64 *ends, u64 slot0, DevState *st, cudaStream_t s) {
    u64 blocks = (n + 255) / 256;
    if (blocks == 0) blocks = 1;
    if (blocks > (u64)num_sms() * 16) blocks = (u64)num_sms() * 16;
    mark_ends_kernel<<<(unsigned)blocks, 256, 0, s>>>(d_offsets, n, off0, nb_total, pad_nb, ends, slot0, st);
}

void launch_count_windows(const u64 *ends, u64 n_slots, u32 k, DevState *st, cudaStream_t s) {
    u64 ngroups = n_slots / 32;
    if (ngroups == 0) return;
    u64 blocks = (ngroups + 255) / 256;
    if (blocks > (u64)num_sms() * 16) blocks = (u64)num_sms() * 16;
    count_windows_kernel<<<(unsigned)blocks, 256, 0, s>>>(ends, n_slots, k, st);
}

}  // namespace sdbg

// radix.cu — step a3: the sorter. "the bottleneck is sorting a set of (k+1)-mers ... in reverse
// lexicographical order of their length-k prefixes" (§2 ¶2). With the key encoding of include/sdbg.h that
// order is the ascending unsigned order of a 2(k+1)-bit integer, so the sort is a least-significant-digit radix sort
// over the significant bits only: P = sum over words of ceil(sigbits/8) stable 8-bit passes.
//
// Each pass is ONE kernel in the onesweep style (the paper's CX1-derived GPU sorter, is prior art, not
// the blueprint): global digit histograms are known up front (fused into the extractor), a tile of keys is ranked
// in shared memory (per-warp digit histograms + warp match ranking, stable in tile order), the tile's digit
// counts are chained to its predecessors by decoupled look-back on 64-bit status words (counts can exceed 2^32:
// config 3 has 3.2e9 records, config 5 31.6e9), and keys are staged bin-sorted in shared memory so that every
// digit's run leaves the SM as one coalesced segment. Tiles are ordered by an atomic ticket, which guarantees that
// every predecessor a tile waits on is already resident (forward progress).
//
// HBM traffic per pass: read n*K + write n*K bytes (K = 8w) — the algorithmic 2nK of DESIGN.md "Byte model" — plus
// 2 KiB of look-back state per tile.
#include "kernels.cuh"

namespace sdbg {

// How step j of a warp finds the lanes holding the same digit ("match"), one letter per step, repeated cyclically:
//   B  8 ballots (VOTE + predicated NOT + AND per bit): ~29 ALU-pipe instructions, no shared memory;
//   A  atomicOr of the lane bit into a warp-private mask word, read back, leader clears: 5 shared-memory
//      operations, ~3 ALU instructions;
//   M  the hardware match.any (one instruction, ~61 SM-cycles per warp on sm_100: only worth a small share).
// The kernel is bound by instruction issue and shared-memory wavefronts at the same time,
// so the steps are split between B and A to load both pipes equally.
#ifndef SDBG_LB_EVERY
#define SDBG_LB_EVERY 4      // rank steps between two look-back polls (power of two)
#endif
#ifndef SDBG_PERSISTENT
#define SDBG_PERSISTENT 1    // 1: persistent CTAs holding the ticket of their next tile; 0: one tile per CTA
#endif
#ifndef SDBG_RANK_METHODS
#define SDBG_RANK_METHODS "BBBBBM"
#endif

template <int W, bool HAS_VAL> struct RadixCfg;
// THREADS x KPT records per tile; keys are staged in shared memory (TILE * 8W bytes).
#ifndef SDBG_R1_THREADS
#define SDBG_R1_THREADS 384   // 384 x 21 = 8,064 keys per tile, 2 CTAs per SM, up to 80 registers (measured best)
#define SDBG_R1_KPT 21
#define SDBG_R1_MINB 2
#endif
template <> struct RadixCfg<1, false> { static constexpr int THREADS = SDBG_R1_THREADS, KPT = SDBG_R1_KPT, MINB = SDBG_R1_MINB; };
template <> struct RadixCfg<2, false> { static constexpr int THREADS = 512, KPT = 8,  MINB = 2; };
template <> struct RadixCfg<3, false> { static constexpr int THREADS = 512, KPT = 5,  MINB = 2; };
#ifndef SDBG_R4_THREADS
#define SDBG_R4_THREADS 256   // 256 x 8 four-word keys = 64 KiB per tile (measured best on config 4)
#define SDBG_R4_KPT 8
#define SDBG_R4_MINB 2
#endif
template <> struct RadixCfg<4, false> { static constexpr int THREADS = SDBG_R4_THREADS, KPT = SDBG_R4_KPT, MINB = SDBG_R4_MINB; };
#ifndef SDBG_R1V_THREADS
#define SDBG_R1V_THREADS 384   // (key word, u32 payload): 384 x 14 (measured best on the pair passes of config 4)
#define SDBG_R1V_KPT 14
#define SDBG_R1V_MINB 2
#endif
template <> struct RadixCfg<1, true>  { static constexpr int THREADS = SDBG_R1V_THREADS, KPT = SDBG_R1V_KPT, MINB = SDBG_R1V_MINB; };
template <> struct RadixCfg<2, true>  { static constexpr int THREADS = 512, KPT = 6,  MINB = 2; };
template <> struct RadixCfg<3, true>  { static constexpr int THREADS = 512, KPT = 4,  MINB = 2; };
template <> struct RadixCfg<4, true>  { static constexpr int THREADS = 512, KPT = 3,  MINB = 2; };

constexpr char kRankMethods[] = SDBG_RANK_METHODS;
constexpr int kNumRankMethods = (int)sizeof(kRankMethods) - 1;
static_assert(kNumRankMethods >= 1 && kNumRankMethods <= 32, "SDBG_RANK_METHODS: 1..32 letters");
constexpr u64 pack_rank_methods() {   // 2 bits per step: 0 = B, 1 = A, 2 = M
    u64 v = 0;
    for (int j = 0; j < kNumRankMethods; ++j)
        v |= (u64)(kRankMethods[j] == 'A' ? 1 : kRankMethods[j] == 'M' ? 2 : 0) << (2 * j);
    return v;
}
constexpr u64 kRankMethodBits = pack_rank_methods();
constexpr int kMethodA = 1, kMethodM = 2;   // 0 = B
__host__ __device__ constexpr int rank_method(int j) { return (int)((kRankMethodBits >> (2 * (j % kNumRankMethods))) & 3u); }
constexpr bool uses_method(int c, int kpt) {
    for (int j = 0; j < kpt; ++j) if (rank_method(j) == c) return true;
    return false;
}

// generic digit of a pass (histogram helpers; the sort kernel uses digit8)
template <int W>
__device__ __forceinline__ u32 digit_of(const u64 (&key)[W], const PassDesc pd) {
    u64 kw = key[0];
#pragma unroll
    for (int j = 1; j < W; ++j) if (pd.word == j) kw = key[j];
    return (u32)(kw >> pd.shift) & ((1u << pd.bits) - 1u);
}

// Digit of a byte-aligned 8-bit pass: byte (psel & 3) of the high (HI) or low half of key word `word`; one PRMT.
template <int W, bool HI>
__device__ __forceinline__ u32 digit8(const u64 (&key)[W], u32 word, u32 psel) {
    u64 kw = key[0];
#pragma unroll
    for (int j = 1; j < W; ++j) if (word == (u32)j) kw = key[j];
    return __byte_perm(HI ? (u32)(kw >> 32) : (u32)kw, 0u, psel);
}

// lanes of the warp whose 8-bit digit equals mine: per bit one ballot, inverted by the lanes whose bit is clear,
// and the eight masks ANDed three at a time (R2P/LOP3 -> predicates, 8 VOTE, 8 predicated NOT, 4 LOP3).
__device__ __forceinline__ u32 match_ballot(u32 d) {
    u32 b[kRadixBits];
#pragma unroll
    for (int i = 0; i < kRadixBits; ++i) {
        asm("{\n\t.reg .pred p;\n\t.reg .b32 t;\n\t"
            "and.b32 t, %1, %2;\n\tsetp.ne.u32 p, t, 0;\n\t"
            "vote.sync.ballot.b32 %0, p, 0xffffffff;\n\t"
            "@!p not.b32 %0, %0;\n\t}" : "=r"(b[i]) : "r"(d), "r"(1u << i));
    }
    u32 m0, m1, m2;
    asm("lop3.b32 %0, %1, %2, %3, 0x80;" : "=r"(m0) : "r"(b[0]), "r"(b[1]), "r"(b[2]));
    asm("lop3.b32 %0, %1, %2, %3, 0x80;" : "=r"(m1) : "r"(b[3]), "r"(b[4]), "r"(b[5]));
    asm("lop3.b32 %0, %1, %2, %3, 0x80;" : "=r"(m2) : "r"(b[6]), "r"(b[7]), "r"(m0));
    return m1 & m2;
}

template <int W>
__device__ __forceinline__ void load_rec(const u64 *__restrict__ src, u64 (&k)[W]) {
    if constexpr (W == 1) {
        k[0] = ld_stream(src);
    } else if constexpr (W == 2) {
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
__device__ __forceinline__ void store_rec(u64 *__restrict__ o, const u64 (&k)[W]) {
    if constexpr (W == 1) {
        o[0] = k[0];
    } else if constexpr (W == 2) {
        *reinterpret_cast<ulonglong2 *>(o) = make_ulonglong2(k[0], k[1]);
    } else if constexpr (W == 4) {
        *reinterpret_cast<ulonglong2 *>(o) = make_ulonglong2(k[0], k[1]);
        *reinterpret_cast<ulonglong2 *>(o + 2) = make_ulonglong2(k[2], k[3]);
    } else {
#pragma unroll
        for (int q = 0; q < W; ++q) o[q] = k[q];
    }
}

// One non-blocking step of the decoupled look-back of one bin (see phase 3 of onesweep_kernel).
// Entry of (tile u, bin) = tag (status, epoch) in bits 63..54, span s in bits 53..32, 32-bit count v in bits 31..0:
//   LOCAL : v = keys of this bin in tiles (u-s, u]   (s = 1 when first published: the tile's own count)
//   GLOBAL: v = keys of this bin in tiles [0, u]
// A walker consumes the entry it requested earlier if it has been published for this pass, jumps over the whole
// span it covers, RE-PUBLISHES its own entry with the span it has covered so far (so later tiles jump over it in
// one step: pointer doubling, the walk is logarithmic in the distance to the nearest GLOBAL entry instead of
// linear), and requests the next entry. On reaching a GLOBAL entry it publishes its inclusive prefix.
// Two layouts of the word: ranges of fewer than 2^32 records (every benchmarked single-range config) keep 32-bit counts
// and 32-bit arithmetic in the walker; larger ranges (block-wise passes over a big workspace) use 34-bit counts.
template <bool WIDE> struct LbFmt;
template <> struct LbFmt<false> {   // [63:62] status [61:54] epoch [53:32] span [31:0] count
    using cnt_t = u32;
    static constexpr int kEpochBits = 8, kTagShift = 54, kSpanShift = 32;
    static constexpr u64 kCntMask = 0xffffffffull;
};
template <> struct LbFmt<true> {    // [63:62] status [61:56] epoch [55:34] span [33:0] count
    using cnt_t = u64;
    static constexpr int kEpochBits = 6, kTagShift = 56, kSpanShift = 34;
    static constexpr u64 kCntMask = (1ull << 34) - 1ull;
};
constexpr u32 kSpanMask = (1u << 22) - 1u;
constexpr u64 kMaxTilesPerRange = 1ull << 22, kMaxRecordsWide = (1ull << 34) - 1ull;

template <bool WIDE>
__device__ __forceinline__ void lookback_poll(u64 *lb, u32 tile, u32 &t, u64 &pend, typename LbFmt<WIDE>::cnt_t &excl, bool &done,
                                              u32 real_cnt, u32 tagL, u32 tagG) {
    using F = LbFmt<WIDE>;
    if (done) return;
    const u32 tag = (u32)(pend >> F::kTagShift);
    if (tag == tagL || tag == tagG) {
        excl += (typename F::cnt_t)(pend & F::kCntMask);
        if (tag == tagG) {
            done = true;
            st_relaxed(lb + (u64)tile * kRadix, ((u64)tagG << F::kTagShift) | (u64)(excl + real_cnt));
            return;
        }
        t -= (u32)(pend >> F::kSpanShift) & kSpanMask;   // tile 0 always publishes GLOBAL, so t never passes it
        st_relaxed(lb + (u64)tile * kRadix, ((u64)tagL << F::kTagShift) | ((u64)(tile - t) << F::kSpanShift) | (u64)(excl + real_cnt));
    }
    pend = ld_relaxed(lb + (u64)t * kRadix);
}

// digit8 that the compiler may not merge with an earlier evaluation (recomputing one PRMT is cheaper than keeping
// 16 digits alive across the phases, which spills)
__device__ __forceinline__ u32 prmt_opaque(u32 x, u32 psel) {
    u32 d;
    asm volatile("prmt.b32 %0, %1, 0, %2;" : "=r"(d) : "r"(x), "r"(psel));
    return d;
}
template <int W, bool HI>
__device__ __forceinline__ u32 digit8_again(const u64 (&key)[W], u32 word, u32 psel) {
    u64 kw = key[0];
#pragma unroll
    for (int j = 1; j < W; ++j) if (word == (u32)j) kw = key[j];
    return prmt_opaque(HI ? (u32)(kw >> 32) : (u32)kw, psel);
}

template <int W, bool HAS_VAL>
struct RadixSmem {
    using Cfg = RadixCfg<W, HAS_VAL>;
    static constexpr int THREADS = Cfg::THREADS, KPT = Cfg::KPT, WARPS = THREADS / 32, TILE = THREADS * KPT;
    static constexpr bool USE_A = uses_method(kMethodA, KPT);
    static constexpr size_t kKeys = 0;                                             // u64[W][TILE]
    static constexpr size_t kBinAddr = kKeys + (size_t)TILE * W * 8;              // u64[256] byte address of bin run - tile start
    static constexpr size_t kValAddr = kBinAddr + kRadix * 8;                       // u64[256] (HAS_VAL)
    static constexpr size_t kBinInfo = kValAddr + (HAS_VAL ? kRadix * 8 : 0);       // u32[2][256] tile count and tile start of the bins
    static constexpr size_t kPos = kBinInfo + 2 * kRadix * 4;                       // u32[WARPS][256] counts, then tile positions
    static constexpr size_t kMask = kPos + (size_t)WARPS * kRadix * 4;              // u32[WARPS][256] match masks (method A)
    static constexpr size_t kVals = kMask + (USE_A ? (size_t)WARPS * kRadix * 4 : 0);  // u32[TILE] (HAS_VAL)
    static constexpr size_t kBytes = kVals + (HAS_VAL ? (size_t)TILE * 4 : 0);
};

// Loads one tile into registers (lane l, step j -> tile index warp*32*KPT + j*32 + l: coalesced 256-byte rows).
// Slots past the end of the data become all-ones pads: digit 255, last in tile order, so they take the last places.
template <int W, bool HAS_VAL, int KPT>
__device__ __forceinline__ void load_tile(const RadixArgs &a, u64 tile_base, u32 cnt, u32 wbase, u64 (&key)[KPT][W],
                                          u32 (&val)[HAS_VAL ? KPT : 1]) {
    if (cnt == (u32)(KPT * RadixCfg<W, HAS_VAL>::THREADS)) {
#pragma unroll
        for (int j = 0; j < KPT; ++j) {
            load_rec<W>(a.keys_in + (tile_base + wbase + j * 32u) * W, key[j]);
            if constexpr (HAS_VAL) val[j] = a.vals_in[tile_base + wbase + j * 32u];
        }
    } else {
#pragma unroll
        for (int j = 0; j < KPT; ++j) {
            const u32 ti = wbase + j * 32u;
            if (ti < cnt) {
                load_rec<W>(a.keys_in + (tile_base + ti) * W, key[j]);
                if constexpr (HAS_VAL) val[j] = a.vals_in[tile_base + ti];
            } else {
#pragma unroll
                for (int q = 0; q < W; ++q) key[j][q] = ~0ull;
                if constexpr (HAS_VAL) val[j] = 0;
            }
        }
    }
}

// L2 prefetch of a contiguous range by the TMA unit (one instruction; bytes a multiple of 16, p 16-byte aligned).
__device__ __forceinline__ void prefetch_l2_bulk(const void *p, u32 bytes) {
    if (bytes) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// Staging of a record in shared memory at tile place pos: one-word keys as u64[TILE]; keys of an even number of words as
// 16-byte halves, half h at ((ulonglong2 *)base)[h * TILE + pos] (one 128-bit access per two words: half the shared-memory
// wavefronts of word-wise accesses at random places); three words word by word.
template <int W, int TILE>
__device__ __forceinline__ void stage_put(u64 *base, u32 pos, const u64 (&k)[W]) {
    if constexpr (W == 2 || W == 4) {
        ulonglong2 *b2 = reinterpret_cast<ulonglong2 *>(base);
#pragma unroll
        for (int h = 0; h < W / 2; ++h) b2[h * TILE + pos] = make_ulonglong2(k[2 * h], k[2 * h + 1]);
    } else {
#pragma unroll
        for (int q = 0; q < W; ++q) base[q * TILE + pos] = k[q];
    }
}
template <int W, int TILE>
__device__ __forceinline__ void stage_get(const u64 *base, u32 pos, u64 (&k)[W]) {
    if constexpr (W == 2 || W == 4) {
        const ulonglong2 *b2 = reinterpret_cast<const ulonglong2 *>(base);
#pragma unroll
        for (int h = 0; h < W / 2; ++h) { const ulonglong2 v = b2[h * TILE + pos]; k[2 * h] = v.x; k[2 * h + 1] = v.y; }
    } else {
#pragma unroll
        for (int q = 0; q < W; ++q) k[q] = base[q * TILE + pos];
    }
}

// One LSD pass over an 8-bit, byte-aligned digit. Persistent CTAs; tiles are handed out by an atomic ticket, one
// tile AHEAD: while a CTA works on a tile it already holds the ticket of its next one, has asked the TMA unit to
// prefetch that tile into L2, and loads it into the (then free) key registers before the write-out of the current
// tile, so that DRAM reads are in flight during the whole life of a tile and not only at its start.
// Per tile:
//   1 count digits of the keys in registers into warp-private histograms (shared atomics);
//   2 one thread per bin: tile count -> look-back state (LOCAL), exclusive scan over bins and warps turns the
//     histograms into the tile position of the first key of (warp, digit);
//   3 per step: match the lanes with my digit, position = running (warp, digit) position + rank among them,
//     key goes to its bin-sorted place in shared memory; the decoupled look-back of the bins advances one
//     predecessor per step in the shadow of the match arithmetic;
//   4 the next tile is loaded into the key registers; bin addresses from the look-back result;
//   5 write-out: place p of the tile goes to bin_address[digit] + p, coalesced per digit run.
// Forward progress: a CTA's current tile is always older than the ticket it holds in reserve, so the oldest
// unfinished tile is always being worked on by a resident CTA.
// FIRST: the first pass of a sort. Its input order is arbitrary, so the pass need not be stable: the rank of a key
// inside (warp, digit) is what the count atomic returned, and the match step of phase 3 is not needed (full tiles
// only: the pads of the last tile rely on the stable order).
template <int W, bool HAS_VAL, bool HI, bool WIDE, bool FIRST = false, bool MAYBE = false>
__global__ void __launch_bounds__(RadixCfg<W, HAS_VAL>::THREADS, RadixCfg<W, HAS_VAL>::MINB)
onesweep_kernel(RadixArgs a) {
    using L = RadixSmem<W, HAS_VAL>;
    using F = LbFmt<WIDE>;
    constexpr int THREADS = L::THREADS, KPT = L::KPT, WARPS = L::WARPS, TILE = L::TILE;
    constexpr bool USE_A = L::USE_A;
    static_assert(THREADS >= kRadix, "one thread per bin");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    u64 *s_keys = reinterpret_cast<u64 *>(smem_raw + L::kKeys);
    u64 *s_binaddr = reinterpret_cast<u64 *>(smem_raw + L::kBinAddr);
    u64 *s_valaddr = reinterpret_cast<u64 *>(smem_raw + L::kValAddr);
    u32 *s_real = reinterpret_cast<u32 *>(smem_raw + L::kBinInfo), *s_bstart = s_real + kRadix;
    u32 *s_pos = reinterpret_cast<u32 *>(smem_raw + L::kPos);
    u32 *s_mask = reinterpret_cast<u32 *>(smem_raw + L::kMask);
    u32 *s_vals = reinterpret_cast<u32 *>(smem_raw + L::kVals);
    __shared__ u32 s_tick[2];
    __shared__ u32 s_wtot[kRadix / 32];

    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const u32 lt = lanemask_lt();
    const u32 word = a.pass.word;
    const u32 psel = 0x4440u | ((a.pass.shift >> 3) & 3u);
    const u32 ntiles = (u32)((a.n + TILE - 1) / TILE);
    const u32 wbase = warp * 32u * KPT + lane;
    u32 *wp = s_pos + warp * kRadix;
    u32 *wm = s_mask + warp * kRadix;
    const u32 tagL = ((u32)kStLocal << F::kEpochBits) | a.epoch, tagG = ((u32)kStGlobal << F::kEpochBits) | a.epoch;
    // two roles of one thread per bin: the first 256 threads scan the histograms, the LAST 256 run the look-back,
    // so that the two chains of dependent shared / L2 round trips proceed side by side
    const bool scanner = tid < kRadix, walker = tid >= THREADS - kRadix;
    u64 *lb = a.lookback + (walker ? tid - (THREADS - kRadix) : tid);   // scanners publish LOCAL of their own bin
    const u32 wbin = tid - (THREADS - kRadix);

    // warp-private histogram rows start at zero (and are zeroed again by their warp after every rank phase)
    auto zero_rows = [&]() {
#pragma unroll
        for (int i = 0; i < kRadix / 32; ++i) {
            wp[i * 32 + lane] = 0;
            if (USE_A) wm[i * 32 + lane] = 0;
        }
        __syncwarp();
    };
    // ---- pieces of the per-tile pipeline ----------------------------------------------------------------------
    u64 key[KPT][W];
    u32 val[HAS_VAL ? KPT : 1];
    u32 it = 0;
    // ticket of the tile after `the one being loaded`, and its L2 prefetch (thread 0)
    auto reserve_next = [&]() {
        if (SDBG_PERSISTENT && tid == 0) {
            const u32 nx = atomicAdd(a.ticket, 1u);
            s_tick[(it + 1) & 1] = nx;
            if (nx < ntiles) {
                const u64 nb = (u64)nx * TILE;
                const u64 nc = (a.n - nb < (u64)TILE) ? a.n - nb : (u64)TILE;
                prefetch_l2_bulk(a.keys_in + nb * W, (u32)(nc * 8u * W) & ~15u);
                if constexpr (HAS_VAL) prefetch_l2_bulk(a.vals_in + nb, (u32)(nc * 4u) & ~15u);
            }
        }
    };
    auto tile_count = [&](u32 t) { return (a.n - (u64)t * TILE < (u64)TILE) ? (u32)(a.n - (u64)t * TILE) : (u32)TILE; };
    // phase 1: digits of the keys in registers -> warp-private histogram
    // MAYBE: a later pass of a sort whose equal keys are merged afterwards (RadixArgs::sorted_lo). The order of equal digits
    // matters only where the bits sorted so far differ; a full tile whose first and last key agree in them (the input is
    // sorted by them, so all its keys do) is ranked like FIRST, the others the stable way.
    constexpr bool RK = FIRST || MAYBE;
    u32 rkp[RK ? (KPT + 1) / 2 : 1];      // arrival rank inside (warp, digit), 16 bits each
    bool uni = false;                     // the tile counted last is ranked by arrival
    auto tile_free = [&](u32 t, u32 c) -> bool {
        if (c != (u32)TILE) return false;                 // the pads of the last tile rely on the stable order
        if constexpr (FIRST) return true;
        const u64 kf = a.keys_in[(u64)t * TILE * W], kl = a.keys_in[((u64)t * TILE + TILE - 1) * W];
        return (((kf ^ kl) >> a.sorted_lo) << (64u - (a.pass.shift - a.sorted_lo))) == 0;   // bits [sorted_lo, pass.shift) agree
    };
    auto count_keys = [&]() {
        if constexpr (RK) {
            if (uni) {
#pragma unroll
                for (int j = 0; j < KPT; ++j) {
                    const u32 r = atomicAdd(&wp[digit8<W, HI>(key[j], word, psel)], 1u);
                    if (j & 1) rkp[j / 2] |= r << 16; else rkp[j / 2] = r;
                }
                return;
            }
        }
#pragma unroll
        for (int j = 0; j < KPT; ++j) atomicAdd(&wp[digit8<W, HI>(key[j], word, psel)], 1u);
    };
    // phase 2a (one thread per bin, after a block barrier): tile count, published LOCAL at once; scan over the bins
    u32 my_cnt = 0, incl = 0;
    auto scan_bins = [&](u32 t, u32 tcnt) {
        my_cnt = 0;
#pragma unroll
        for (int v = 0; v < WARPS; ++v) my_cnt += s_pos[v * kRadix + tid];
        u32 rc = my_cnt;                                                  // my_cnt includes the pads (bin 255)
        if (tid == kRadix - 1) rc -= (u32)TILE - tcnt;
        st_relaxed(a.lookback + tid + (u64)t * kRadix, ((u64)(t == 0 ? tagG : tagL) << F::kTagShift) | (t == 0 ? 0ull : 1ull << F::kSpanShift) | rc);
        s_real[tid] = rc;
        incl = warp_incl_scan_add(my_cnt);
        if (lane == 31) s_wtot[warp] = incl;
    };
    // phase 2b (after another barrier): entry (v, bin) becomes the tile position of the first key of digit `bin`
    // held by warp v; returns the tile position of the bin's first key
    auto scan_warps = [&]() {
        u32 off = 0;
#pragma unroll
        for (int w = 0; w < kRadix / 32; ++w) off += (w < (int)warp) ? s_wtot[w] : 0u;
        const u32 bs = off + incl - my_cnt;
        u32 run = bs;
#pragma unroll
        for (int v = 0; v < WARPS; ++v) {
            const u32 t = s_pos[v * kRadix + tid];
            s_pos[v * kRadix + tid] = run;
            run += t;
        }
        s_bstart[tid] = bs;
    };

    // Decoupled look-back state of the CURRENT tile, one thread per bin. It advances during the rank steps of the
    // tile and, in the shadow of the next tile's count and scan, until the write-out needs it. lb_t = predecessor
    // tile being examined; lb_pend = its entry as last read.
    u64 lb_pend = 0;
    typename F::cnt_t lb_excl = 0;
    u32 lb_t = 0, real_cnt = 0, bin_start = 0;
    bool lb_done = true;
    auto lookback_begin = [&](u32 t) {   // after the barrier that follows scan_warps of tile t
        real_cnt = s_real[wbin];
        bin_start = s_bstart[wbin];
        lb_excl = 0;
        lb_done = true;
        if (t != 0) {
            lb_done = false;
            lb_t = t - 1;
            lb_pend = ld_relaxed(lb + (u64)lb_t * kRadix);
        }
    };

    // ---- prologue: first tile up to the point where its (warp, digit) positions are known ---------------------------
    if (tid == 0) s_tick[0] = atomicAdd(a.ticket, 1u);
    zero_rows();
    __syncthreads();
    u32 tile = s_tick[0];
    if (tile >= ntiles) return;
    u32 cnt = tile_count(tile);
    load_tile<W, HAS_VAL, KPT>(a, (u64)tile * TILE, cnt, wbase, key, val);
    reserve_next();
    if constexpr (RK) uni = tile_free(tile, cnt);
    count_keys();
    __syncthreads();
    if (scanner) scan_bins(tile, cnt);
    __syncthreads();
    if (scanner) scan_warps();
    __syncthreads();
    if (walker) lookback_begin(tile);

    for (;; ++it) {
        const u32 next = SDBG_PERSISTENT ? s_tick[(it + 1) & 1] : ntiles;
        // ---- 3: rank within the warp (stable in tile order), scatter to shared memory in bin-sorted order ------
        bool ranked = false;
        if constexpr (RK) {
            if (uni) {
                ranked = true;
#pragma unroll
                for (int j = 0; j < KPT; ++j) {
                    const u32 d = digit8_again<W, HI>(key[j], word, psel);
                    const u32 pos = wp[d] + ((rkp[j / 2] >> (16 * (j & 1))) & 0xffffu);
                    stage_put<W, TILE>(s_keys, pos, key[j]);
                    if constexpr (HAS_VAL) s_vals[pos] = val[j];
                    if ((j & (SDBG_LB_EVERY - 1)) == SDBG_LB_EVERY - 1 && walker)
                        lookback_poll<WIDE>(lb, tile, lb_t, lb_pend, lb_excl, lb_done, real_cnt, tagL, tagG);
                }
                __syncwarp();
            }
        }
        if (!ranked) {
#pragma unroll
        for (int j = 0; j < KPT; ++j) {
            const u32 d = digit8_again<W, HI>(key[j], word, psel);
            const int method = rank_method(j);                        // constant after unrolling
            u32 m;
            if (method == kMethodA) {
                atomicOr(&wm[d], 1u << lane);
                __syncwarp();
                m = wm[d];
            } else if (method == kMethodM) {
                m = __match_any_sync(0xffffffffu, d);
            } else {
                m = match_ballot(d);
            }
            const u32 prev = wp[d];                                   // same address within the group: broadcast read
            __syncwarp();
            if ((m >> lane) <= 1u) {                                  // highest lane of the group
                wp[d] = prev + __popc(m);
                if (method == kMethodA) wm[d] = 0;
            }
            const u32 pos = prev + __popc(m & lt);
            stage_put<W, TILE>(s_keys, pos, key[j]);
            if constexpr (HAS_VAL) s_vals[pos] = val[j];
            __syncwarp();
            if ((j & (SDBG_LB_EVERY - 1)) == SDBG_LB_EVERY - 1 && walker)
                lookback_poll<WIDE>(lb, tile, lb_t, lb_pend, lb_excl, lb_done, real_cnt, tagL, tagG);
        }
        }
        zero_rows();   // own rows only; their last readers were the scan threads, two barriers ago

        // ---- 1', 2' of the NEXT tile, with the look-back of the current one advancing behind them ------------------
        const u32 cur_cnt = cnt;
        if (next < ntiles) {
            cnt = tile_count(next);
            load_tile<W, HAS_VAL, KPT>(a, (u64)next * TILE, cnt, wbase, key, val);
            ++it; reserve_next(); --it;
            if constexpr (RK) uni = tile_free(next, cnt);
            count_keys();
        }
        __syncthreads();
        if (scanner && next < ntiles) scan_bins(next, cnt);
        if (walker) lookback_poll<WIDE>(lb, tile, lb_t, lb_pend, lb_excl, lb_done, real_cnt, tagL, tagG);
        __syncthreads();
        if (scanner && next < ntiles) scan_warps();
        if (walker) {
            // ---- 4: the look-back result is needed now -------------------------------------------------------------
            while (!lb_done) lookback_poll<WIDE>(lb, tile, lb_t, lb_pend, lb_excl, lb_done, real_cnt, tagL, tagG);
            const u64 first = a.bin_base[wbin] + lb_excl - bin_start;   // output index of tile place 0 if it were in this bin
            s_binaddr[wbin] = reinterpret_cast<u64>(a.keys_out) + first * (8ull * W);
            if constexpr (HAS_VAL) s_valaddr[wbin] = reinterpret_cast<u64>(a.vals_out) + first * 4ull;
        }
        __syncthreads();
        if (walker && next < ntiles) lookback_begin(next);

        // ---- 5: coalesced write-out: place p of the tile goes to bin address[digit] + p ----------------------------
        auto write_place = [&](u32 p) {
            u64 kk[W];
            stage_get<W, TILE>(s_keys, p, kk);
            const u32 d = digit8<W, HI>(kk, word, psel);
            store_rec<W>(reinterpret_cast<u64 *>(s_binaddr[d] + (u64)p * (8u * W)), kk);
            if constexpr (HAS_VAL) *reinterpret_cast<u32 *>(s_valaddr[d] + (u64)p * 4u) = s_vals[p];
        };
        if (cur_cnt == (u32)TILE) {
#pragma unroll
            for (int i = 0; i < KPT; ++i) write_place(i * THREADS + tid);
        } else {
#pragma unroll 1
            for (u32 p = tid; p < cur_cnt; p += THREADS) write_place(p);
        }
        if (next >= ntiles) break;
        tile = next;
        __syncthreads();   // s_keys is rewritten by the rank steps that follow
    }
}

template <int W, bool HAS_VAL>
static int setup_one() {
    const int bytes = (int)RadixSmem<W, HAS_VAL>::kBytes;
    if constexpr (W == 1 || (W == 2 && !HAS_VAL)) {      // the unstable variants (narrow look-back words)
        int e2;
        if ((e2 = (int)cudaFuncSetAttribute(onesweep_kernel<W, HAS_VAL, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes))) return e2;
        if ((e2 = (int)cudaFuncSetAttribute(onesweep_kernel<W, HAS_VAL, true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes))) return e2;
        if ((e2 = (int)cudaFuncSetAttribute(onesweep_kernel<W, HAS_VAL, false, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes))) return e2;
        if ((e2 = (int)cudaFuncSetAttribute(onesweep_kernel<W, HAS_VAL, true, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes))) return e2;
    }
    int e = (int)cudaFuncSetAttribute(onesweep_kernel<W, HAS_VAL, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e) return e;
    e = (int)cudaFuncSetAttribute(onesweep_kernel<W, HAS_VAL, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e || HAS_VAL) return e;   // ranges of 2^32 records and more exist only in sdbg_count_edges (keys without payload)
    if constexpr (W == 1) {
        e = (int)cudaFuncSetAttribute(onesweep_kernel<1, false, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e) return e;
        e = (int)cudaFuncSetAttribute(onesweep_kernel<1, false, true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e) return e;
        e = (int)cudaFuncSetAttribute(onesweep_kernel<1, false, false, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e) return e;
        e = (int)cudaFuncSetAttribute(onesweep_kernel<1, false, true, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e) return e;
        e = (int)cudaFuncSetAttribute(onesweep_kernel<1, false, false, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e) return e;
        e = (int)cudaFuncSetAttribute(onesweep_kernel<1, false, true, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e) return e;
        e = (int)cudaFuncSetAttribute(onesweep_kernel<1, false, false, true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e) return e;
        e = (int)cudaFuncSetAttribute(onesweep_kernel<1, false, true, true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e) return e;
    }
    e = (int)cudaFuncSetAttribute(onesweep_kernel<W, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e) return e;
    return (int)cudaFuncSetAttribute(onesweep_kernel<W, false, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

int radix_setup() {
    int e = 0;
    if ((e = setup_one<1, false>())) return e;
    if ((e = setup_one<2, false>())) return e;
    if ((e = setup_one<3, false>())) return e;
    if ((e = setup_one<4, false>())) return e;
    if ((e = setup_one<1, true>())) return e;
    if ((e = setup_one<2, true>())) return e;
    if ((e = setup_one<3, true>())) return e;
    if ((e = setup_one<4, true>())) return e;
    return 0;
}

template <int W, bool HAS_VAL>
static constexpr u64 tile_of() { return (u64)RadixCfg<W, HAS_VAL>::THREADS * RadixCfg<W, HAS_VAL>::KPT; }

// most records one sort may hold: 22-bit spans (tiles) and 34-bit counts in the look-back words; payloads: 32-bit counts
u64 radix_max_records(u32 W, bool v) {
    const u64 by_tiles = kMaxTilesPerRange * radix_tile_records(W, v);
    const u64 by_count = v ? 0xffffffffull : kMaxRecordsWide;
    return by_tiles < by_count ? by_tiles : by_count;
}

u64 radix_tile_records(u32 W, bool v) {
    switch (W) {
        case 1: return v ? tile_of<1, true>() : tile_of<1, false>();
        case 2: return v ? tile_of<2, true>() : tile_of<2, false>();
        case 3: return v ? tile_of<3, true>() : tile_of<3, false>();
        case 4: return v ? tile_of<4, true>() : tile_of<4, false>();
    }
    return 0;
}

static u64 g_unstable_launches = 0;
u64 radix_unstable_launches() { return g_unstable_launches; }

template <int W, bool HAS_VAL>
static int launch_one(const RadixArgs &a, cudaStream_t s) {
    const u64 tiles = (a.n + tile_of<W, HAS_VAL>() - 1) / tile_of<W, HAS_VAL>();
    if (tiles == 0) return 0;
    if (tiles > kMaxTilesPerRange || a.n > kMaxRecordsWide) return (int)cudaErrorInvalidValue;   // look-back word layout
    const bool wide = a.n > 0xffffffffull || (a.force_wide && !HAS_VAL);
    if (wide && HAS_VAL) return (int)cudaErrorInvalidValue;
    if (a.pass.bits != kRadixBits || (a.pass.shift & 7u)) return (int)cudaErrorInvalidValue;   // byte-aligned digits only
    // persistent CTAs: every SM filled to the occupancy the kernel was built for
    const u64 resident = SDBG_PERSISTENT ? (u64)num_sms() * RadixCfg<W, HAS_VAL>::MINB : tiles;
    const unsigned g = (unsigned)(tiles < resident ? tiles : resident), t = RadixCfg<W, HAS_VAL>::THREADS;
    const size_t sm = RadixSmem<W, HAS_VAL>::kBytes;
    const bool hi = a.pass.shift >= 32;
    if constexpr (!HAS_VAL) {
        if (wide) {
            if constexpr (W == 1) {                      // the same two unstable variants with wide look-back words
                if (a.unstable) {
                    ++g_unstable_launches;
                    if (hi) onesweep_kernel<1, false, true, true, true><<<g, t, sm, s>>>(a);
                    else    onesweep_kernel<1, false, false, true, true><<<g, t, sm, s>>>(a);
                    return (int)cudaGetLastError();
                }
                if (a.maybe_unstable && a.sorted_lo < a.pass.shift) {
                    ++g_unstable_launches;
                    if (hi) onesweep_kernel<1, false, true, true, false, true><<<g, t, sm, s>>>(a);
                    else    onesweep_kernel<1, false, false, true, false, true><<<g, t, sm, s>>>(a);
                    return (int)cudaGetLastError();
                }
            }
            if (hi) onesweep_kernel<W, false, true, true><<<g, t, sm, s>>>(a);
            else    onesweep_kernel<W, false, false, true><<<g, t, sm, s>>>(a);
            return (int)cudaGetLastError();
        }
    }
    // one-word keys (with or without payload: the stand-in pairs of long keys) and two-word records: the unstable variants
    if constexpr (W == 1 || (W == 2 && !HAS_VAL)) {
        if (a.unstable) {
            ++g_unstable_launches;
            if (hi) onesweep_kernel<W, HAS_VAL, true, false, true><<<g, t, sm, s>>>(a);
            else    onesweep_kernel<W, HAS_VAL, false, false, true><<<g, t, sm, s>>>(a);
            return (int)cudaGetLastError();
        }
        if (a.maybe_unstable && a.sorted_lo < a.pass.shift && a.pass.word == 0) {
            ++g_unstable_launches;
            if (hi) onesweep_kernel<W, HAS_VAL, true, false, false, true><<<g, t, sm, s>>>(a);
            else    onesweep_kernel<W, HAS_VAL, false, false, false, true><<<g, t, sm, s>>>(a);
            return (int)cudaGetLastError();
        }
    }
    if (hi) onesweep_kernel<W, HAS_VAL, true, false><<<g, t, sm, s>>>(a);
    else    onesweep_kernel<W, HAS_VAL, false, false><<<g, t, sm, s>>>(a);
    return (int)cudaGetLastError();
}

int launch_radix_pass(const RadixArgs &a, cudaStream_t s) {
    const bool v = a.vals_in != nullptr;
    switch (a.W) {
        case 1: return v ? launch_one<1, true>(a, s) : launch_one<1, false>(a, s);
        case 2: return v ? launch_one<2, true>(a, s) : launch_one<2, false>(a, s);
        case 3: return v ? launch_one<3, true>(a, s) : launch_one<3, false>(a, s);
        case 4: return v ? launch_one<4, true>(a, s) : launch_one<4, false>(a, s);
    }
    return (int)cudaErrorInvalidValue;
}

// ---- multi-word keys: word-wise LSD with an index payload -------------------------------------------------------------
// Keys of W > 1 words are not moved through the passes themselves: the sorter moves (one key word, u32 record index)
// pairs with the one-word kernel, least significant word first, and fetches the word of the next level through the
// index; one last gather puts the whole records in order. Per record a pass then moves 2 x 12 bytes instead of
// 2 x 8W, at the price of W + 1 gathers (32-byte sectors). Stable passes make this the same LSD sort.
__global__ void __launch_bounds__(256) gather_word_kernel(const u64 *__restrict__ recs, u32 W, u32 q, const u32 *__restrict__ idx_in,
                                                          u64 *__restrict__ word_out, u32 *__restrict__ idx_out, u64 n) {
    for (u64 j = (u64)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += (u64)gridDim.x * blockDim.x) {
        const u64 i = idx_in ? (u64)idx_in[j] : j;
        word_out[j] = __ldg(recs + i * W + q);
        if (idx_out) idx_out[j] = (u32)i;     // first level: identity
    }
}
template <int W>
__global__ void __launch_bounds__(256) gather_recs_kernel(const u64 *__restrict__ recs, const u32 *__restrict__ idx, u64 *__restrict__ out, u64 n) {
    for (u64 j = (u64)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += (u64)gridDim.x * blockDim.x) {
        u64 k[W];
        load_rec<W>(recs + (u64)idx[j] * W, k);
        store_rec<W>(out + j * W, k);
    }
}
static unsigned gather_blocks(u64 n) {
    u64 b = (n + 255) / 256;
    const u64 cap = (u64)num_sms() * 16;
    return (unsigned)(b < cap ? b : cap);
}
void launch_gather_word(const u64 *recs, u32 W, u32 q, const u32 *idx_in, u64 *word_out, u32 *idx_out, u64 n, cudaStream_t s) {
    if (n) gather_word_kernel<<<gather_blocks(n), 256, 0, s>>>(recs, W, q, idx_in, word_out, idx_out, n);
}
void launch_gather_recs(const u64 *recs, u32 W, const u32 *idx, u64 *out, u64 n, cudaStream_t s) {
    if (!n) return;
    switch (W) {
        case 2: gather_recs_kernel<2><<<gather_blocks(n), 256, 0, s>>>(recs, idx, out, n); break;
        case 3: gather_recs_kernel<3><<<gather_blocks(n), 256, 0, s>>>(recs, idx, out, n); break;
        case 4: gather_recs_kernel<4><<<gather_blocks(n), 256, 0, s>>>(recs, idx, out, n); break;
        default: gather_recs_kernel<1><<<gather_blocks(n), 256, 0, s>>>(recs, idx, out, n); break;
    }
}

// ---- histogram helpers ------------------------------------------------------------------------------------------

// in-place exclusive scan of each pass's 256 u64 bins; one block per pass
__global__ void __launch_bounds__(kRadix) scan_hist_kernel(u64 *hist) {
    __shared__ u64 s_w[kRadix / 32];
    u64 *h = hist + (size_t)blockIdx.x * kRadix;
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const u64 v = h[tid];
    u64 incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        u64 t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= (u32)o) incl += t;
    }
    if (lane == 31) s_w[warp] = incl;
    __syncthreads();
    u64 off = 0;
    for (u32 w = 0; w < warp; ++w) off += s_w[w];
    h[tid] = off + incl - v;
}

void launch_scan_hist(u64 *digit_hist, int n_passes, cudaStream_t s) {
    if (n_passes > 0) scan_hist_kernel<<<n_passes, kRadix, 0, s>>>(digit_hist);
}

// digit histograms of all passes over an existing key array (sdbg_build's unsorted path)
template <int W>
__global__ void __launch_bounds__(256) key_hist_kernel(const u64 *__restrict__ keys, u64 n, PassTable pt, u64 *hist) {
    extern __shared__ u32 s_hist[];
    for (int i = threadIdx.x; i < pt.n * kRadix; i += blockDim.x) s_hist[i] = 0;
    __syncthreads();
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (u64)gridDim.x * blockDim.x) {
        u64 key[W];
#pragma unroll
        for (int q = 0; q < W; ++q) key[q] = keys[i * W + q];
        for (int p = 0; p < pt.n; ++p) atomicAdd(&s_hist[p * kRadix + digit_of<W>(key, pt.p[p])], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < pt.n * kRadix; i += blockDim.x)
        if (s_hist[i]) atomicAdd(&hist[i], (u64)s_hist[i]);
}

void launch_key_hist(const u64 *keys, u64 n, u32 W, const PassTable &pt, u64 *hist, cudaStream_t s) {
    if (n == 0) return;
    u64 blocks = (n + 255) / 256;
    if (blocks > (u64)num_sms() * 8) blocks = (u64)num_sms() * 8;
    size_t smem = (size_t)pt.n * kRadix * 4;
    switch (W) {
        case 1: key_hist_kernel<1><<<(unsigned)blocks, 256, smem, s>>>(keys, n, pt, hist); break;
        case 2: key_hist_kernel<2><<<(unsigned)blocks, 256, smem, s>>>(keys, n, pt, hist); break;
        case 3: key_hist_kernel<3><<<(unsigned)blocks, 256, smem, s>>>(keys, n, pt, hist); break;
        case 4: key_hist_kernel<4><<<(unsigned)blocks, 256, smem, s>>>(keys, n, pt, hist); break;
    }
}

}  // namespace sdbg

// kernels.cuh — launch prototypes of the libsdbg kernels and the device helpers several of them share.
#pragma once
#include "common.cuh"

namespace sdbg {

// Valid-window mask of slots [32g, 32g+32): bit b set iff no end mark lies in [32g+b, 32g+b+k), i.e. the (k+1)-window
// starting there lies inside one read. Reads ends words up to (32g+32+k)/64 (the guard slots keep that in bounds).
__device__ __forceinline__ u32 valid_mask32(const u64 *__restrict__ ends, u64 g, u32 k) {
    const u64 wi = g >> 1;
    const u32 sh = (u32)(g & 1) * 32;
    u64 e0 = __ldg(ends + wi), e1 = __ldg(ends + wi + 1), e2 = 0, e3 = 0;
    if (sh + 31 + k > 128) { e2 = __ldg(ends + wi + 2); }
    if (sh + 31 + k > 192) { e3 = __ldg(ends + wi + 3); }
    u64 v0, v1, v2;
    if (sh) {
        v0 = (e0 >> 32) | (e1 << 32); v1 = (e1 >> 32) | (e2 << 32); v2 = (e2 >> 32) | (e3 << 32);
    } else {
        v0 = e0; v1 = e1; v2 = e2;
    }
    // smear: bit b of v0 becomes OR of original bits b .. b+k-1
    u32 cover = 1;
    while (cover * 2 <= k) {
        v0 |= (v0 >> cover) | (v1 << (64 - cover));
        v1 |= (v1 >> cover) | (v2 << (64 - cover));
        v2 |= (v2 >> cover);
        cover *= 2;
    }
    if (cover < k) {
        const u32 m = k - cover;   // 1..63
        v0 |= (v0 >> m) | (v1 << (64 - m));
    }
    return ~(u32)v0;
}

// ---- launchers (host) ----------------------------------------------------------------------------------
void launch_pack(const unsigned char *d_ascii, u64 nb, u64 *words, u64 slot0, u64 err_index_base, DevState *st, cudaStream_t s);
void launch_mark_ends(const u64 *d_offsets, u64 n, u64 off0, u64 nb_total, u64 pad_nb, u64 *ends, u64 slot0, DevState *st, cudaStream_t s);
void launch_count_windows(const u64 *ends, u64 n_slots, u32 k, DevState *st, cudaStream_t s);

struct ExtractArgs {
    const u64 *words, *ends;
    u64 n_slots;
    u32 k, W;
    u32 bucket_lo, bucket_hi;     // keep keys with bucket in [lo, hi); full range = [0, 65536)
    u64 *keys_out;                // nullptr: histogram-only
    u64 out_cap;                  // records keys_out can hold
    u64 *digit_hist;              // nullptr or u64[n_passes][256], accumulated
    u32 hist_top;                 // != 0: only the rows of the hist_top most significant passes are needed (the others may stay short)
    u64 *bucket_hist;             // nullptr or u64[65536], accumulated (all buckets, ignores lo/hi)
    u64 *coarse_hist;             // nullptr or u64[4096], accumulated: records per group of 16 consecutive l=8 partitions (top 12 key
                                  // bits). Histogram-only call (nothing else set), k >= 8: counted in shared memory, no key is made
    int want_csum;
    PassTable passes;
    // keys of three and four words on the table-count path: beside every record (same index) a sortable stand-in of one word,
    // pair_keys[i] = top pair_top_bits bits of the first key word | fingerprint of the whole key below them (pair_key() in
    // common.cuh), and pair_idx[i] = i. The top passes then move 12 bytes per record instead of 8 W.
    u64 *pair_keys; u32 *pair_idx; u32 pair_top_bits;
    // with pair_keys, dense range: a warp takes the 32 slots of ONE group per step (lane = slot) instead of a lane taking 32
    // consecutive slots: groups without a valid window are skipped warp-wide (at k = 99 on 150 bases a third of the slots
    // start a window, and the lanes of the other mapping idle two steps out of three)
    bool by_rows;
};
int launch_extract(const ExtractArgs &a, DevState *st, cudaStream_t s);

// extraction fused with the first radix pass (extract.cu): one-word keys of a dense range scattered into the 256 bins of
// key byte t (0 = most significant); bin_cursor[b] = first output place of bin b, advanced by the kernel
struct ScatterArgs {
    const u64 *words, *ends;
    u64 n_slots;
    u32 k, t;
    u64 *keys_out; u64 out_cap;
    u64 *bin_cursor;              // u64[256], exclusive prefix of the bin sizes (from the histogram pre-scan)
};
int extract_scatter_setup();
bool extract_scatter_supported(u32 k, u32 t);
int launch_extract_scatter(const ScatterArgs &a, cudaStream_t s);

// exclusive scan of each pass's 256-bin histogram, in place (u64)
void launch_scan_hist(u64 *digit_hist, int n_passes, cudaStream_t s);

struct RadixArgs {
    const u64 *keys_in; u64 *keys_out;
    const u32 *vals_in; u32 *vals_out;   // nullptr: keys only
    u64 n; u32 W;
    const u64 *bin_base;                 // u64[256] exclusive bases of this pass
    u64 *lookback;                       // u64[tiles*256], zeroed once per sort; epoch-tagged per pass
    u32 *ticket;                         // zeroed
    PassDesc pass; u32 epoch;
    bool force_wide;                     // use the layout for ranges of 2^32 records and more whatever n is (tests)
    bool maybe_unstable; u32 sorted_lo;  // a LATER pass of such a sort (same contract as `unstable`, (b) above all): the input is sorted by key
                                         // bits [sorted_lo, pass.shift); tiles whose keys all agree in them are ranked by arrival
    bool unstable;                       // CONTRACT: set only when (a) this is pass 0 of a multi-pass sort whose input order carries no
                                         // information AND (b) the caller merges equal keys afterwards (sdbg_count_edges). The pass then
                                         // need not keep the order of equal digits (radix.cu FIRST: rank = return value of the count atomic,
                                         // hardware-defined among the lanes of a warp). A single pass that refines an existing order
                                         // (api_full.inc compute_zero_degree) must leave it false; launch_radix_pass counts FIRST launches in
                                         // radix_unstable_launches() so that tests can assert who used it.
};
u64 radix_tile_records(u32 W, bool has_vals);
u64 radix_max_records(u32 W, bool has_vals);   // cap of one sort range (look-back word layout)
int launch_radix_pass(const RadixArgs &a, cudaStream_t s);
u64 radix_unstable_launches();           // launches of the FIRST (unstable) variant by this process so far
// multi-word keys (radix.cu "word-wise LSD with an index payload")
void launch_gather_word(const u64 *recs, u32 W, u32 q, const u32 *idx_in, u64 *word_out, u32 *idx_out, u64 n, cudaStream_t s);
void launch_gather_recs(const u64 *recs, u32 W, const u32 *idx, u64 *out, u64 n, cudaStream_t s);
int radix_setup();   // sets max dynamic shared memory attributes; once per process

// keys-only digit histograms over an existing key array (sdbg_build unsorted path)
void launch_key_hist(const u64 *keys, u64 n, u32 W, const PassTable &pt, u64 *digit_hist, cudaStream_t s);

struct CountArgs {
    const u64 *keys; u64 n; u32 W, d;
    u64 *out_keys; u32 *out_mult; u64 out_cap;
    u64 *tile_sums;          // scratch of 8 bytes per count_tile_records() records: u64 per block of the sweeps (solid
                             // edges, then their exclusive prefix), behind them u32 per warp chunk
    u64 *stash;              // scratch of 8 bytes per record (the sorter's spare buffer): the sweep leaves (place in chunk,
                             // multiplicity) of every solid edge there, chunk by chunk
    u64 *stat_slots;         // u64[kStatSlots][kStatSlotWords], accumulated
    int want_csum;
    bool force_wide;         // 64-bit run lengths whatever n is (tests)
    int range_parity;        // reads st->out_cursor[parity], writes st->out_cursor[parity^1]
};
u64 count_tile_records(u32 W);
int launch_count_filter(const CountArgs &a, DevState *st, cudaStream_t s);
// records sorted by their top key bytes only: count in shared-memory tables, segment by segment (hashcount.cu)
constexpr u32 kHashSegBlock = 64;        // segments per block sum
struct HashCountArgs {
    const u64 *keys; u64 n;              // one word per record, sorted by key >> top_shift: the key itself (W = 1) or its
                                         // stand-in (ExtractArgs::pair_keys)
    u32 W;                               // words per record (0 = 1)
    const u32 *vals; const u64 *recs;    // (W > 2) vals[i] = index of the record of keys[i] in recs (W words each, any order).
                                         // W = 2: keys holds the sorted records themselves (2 words each), vals and recs are null
    bool weak_fp;                        // (tests, W = 2) fingerprint = first word
    u32 top_shift, chunk, window;        // nominal records per segment; how far a bucket may run past a nominal border
    u32 d;                               // solid threshold, >= 2
    u64 nseg;                            // ceil(n / chunk)
    u64 *seg_start;                      // u64[nseg + 1] scratch
    u64 *seg_count;                      // u64[nseg] scratch: solid edges per segment
    u32 *seg_list; u32 *n_list;          // null, or u32[nseg] + one word of scratch: the non-empty segments (long buckets)
    u64 *blk_sum;                        // u64[ceil(nseg / 64)] scratch, zeroed: solid edges per block of 64 segments, then their prefix
    u64 *stage_keys;                     // u64[n W] scratch (the sorter's spare buffer, or the second record buffer)
    u32 *ticket;                         // zeroed: segments are handed out in order
    u32 *overflow;                       // zeroed; nonzero afterwards: something did not fit, nothing may be used
    u64 *stat_slots;
    const u64 *cursor_in; u64 *cursor_out;   // solid edges appended before this range / after it (DevState::out_cursor)
    u64 *out_keys; u32 *out_mult; u64 out_cap;
};
int hash_setup();
void launch_hash_bounds(const HashCountArgs &a, cudaStream_t s);
int launch_hash_count(const HashCountArgs &a, cudaStream_t s);
void launch_hash_append(const HashCountArgs &a, u64 *total /* device scratch */, cudaStream_t s);

struct EmitArgs {
    const u64 *keys; const u32 *mult_in; u64 n; u32 k, W;
    uint8_t *Wout; u32 *last_bits32; u32 *mult_out;
};
void launch_emit(const EmitArgs &a, cudaStream_t s);

// lossless extras (dummies.cu): `$` edges, zero-indegree vector, validity bits
struct FullArgs {
    const u64 *keys; const u32 *mult_in; u64 n; u32 k;     // sorted solid edges
    const uint8_t *W_real; const u32 *last_real32;         // their emitted arrays
    const u64 *tk;                                         // sorted target node keys (WT words each)
    const u32 *zout_idx; u64 n_zero_out;                   // indices into tk of the nodes without outgoing edge
    const u32 *zin_idx; u64 t;                             // indices of edges whose node has no incoming edge
    uint8_t *out_W; u32 *out_last32; u64 *out_valid; u32 *out_mult; u64 *aux_bits;
    const uint8_t *flag_in; u32 *out_zin32;                // per solid edge: last edge of a zero-indegree node -> zin bits (A24)
    u64 *F_dev;                                            // u64[4] device scratch: F[0..3] of reading A25
    u32 *dpos;                                             // u32[n_zero_out] scratch: output position of each `$` edge
};
int launch_target_keys(const u64 *keys, u64 n, u32 k, u32 W, u32 WT, u64 *out, cudaStream_t s);
u64 zero_flags_index_bytes(u32 k);   // scratch of the two prefix indices (edges, targets)
int launch_zero_flags(const u64 *keys, u64 n, u32 k, u32 W, u32 WT, const u64 *tk_sorted, const u32 *last_real32,
                      u32 *prefix_index, uint8_t *flag_out, uint8_t *flag_in, cudaStream_t s);
u64 flag_scratch_bytes(u64 n);
void launch_compact_flags(const uint8_t *flag, u64 n, u64 *scratch, u32 *out_idx, u64 *total_out, cudaStream_t s);
int launch_full_assemble(const FullArgs &a, u32 W, u32 WT, cudaStream_t s);

// traversal (rank.cu): rank/select cells over B_A, B_C, B_G, B_T, H and the forward / backward maps
struct IndexView {
    const u64 *cells; u64 n_cells, m;                      // vector v at cells + v * n_cells * 8 words
    u32 *samples[5]; u64 n_samples[5];                     // cell of every 512-th one; (ones + 511) / 512 entries
    u64 F[5], HF[5];                                       // F array (A25) and rank_H(F[c])
    const uint8_t *W; const u64 *last_bits;                // borrowed from the graph
};
u64 index_cells(u64 m);
u64 index_samples_cap(u64 m);
u64 index_scratch_words(u64 m);
void launch_index_build(const uint8_t *W, const u64 *last_bits, const u64 *zin_bits, const IndexView &ix, u64 *scratch /* u64[index_scratch_words(m)] */, cudaStream_t s);
// the same with the scratch in a static device array of rank.cu (no allocation anywhere; m <= index_static_max_edges())
u64 index_static_max_edges();
int launch_index_build_static(const uint8_t *W, const u64 *last_bits, const u64 *zin_bits, const IndexView &ix, u64 **scratch_out, cudaStream_t s);
void launch_forward(const IndexView &ix, const u64 *q, u64 n, long long *out, cudaStream_t s);
void launch_backward(const IndexView &ix, const u64 *q, u64 n, long long *out, cudaStream_t s);

// mercy-kmers (mercy.cu)
struct MercyArgs {
    const u64 *words, *ends; u64 n_slots;                  // packed reads
    const u64 *keys; u64 n; u32 k;                         // sorted solid edges
    const void *table; u64 table_mask;                     // hash table over the solid edges: 16-byte slots {first key word, edge index + 1 (0 = empty)}
    const u64 *tk; const u32 *zout_idx; u64 n_zero_out;    // nodes without outgoing edge (rows of tk)
    const u32 *zin_idx; u64 t;                             // nodes without incoming edge (edges whose node it is)
    u64 *out_keys; u32 *out_mult; u64 out_cap;             // appended at st->extract_cursor
};
void launch_hash_build(const u64 *keys, u64 n, u32 W, void *table /* 16 bytes per slot, zeroed */, u64 slots /* power of two >= 2n */, cudaStream_t s);
int launch_mercy(const MercyArgs &a, u32 W, u32 WT, DevState *st, cudaStream_t s);

// sdbg_build unsorted path: merge equal adjacent keys of a sorted (key, mult) list, summing mult (saturating).
struct MergeArgs {
    const u64 *keys; const u32 *mult; u64 n; u32 W;
    u64 *out_keys; u32 *out_mult;        // capacity n
    u64 *sums;                           // scratch of 8 bytes per merge_tile_records() records (block and chunk sums)
    u64 *acc;                            // u64[n] scratch accumulators, zeroed
};
u64 merge_tile_records();
void launch_merge(const MergeArgs &a, DevState *st, cudaStream_t s);

}  // namespace sdbg

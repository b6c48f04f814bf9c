/* sdbg.h — C ABI of libsdbg: the data-parallel hot path of MEGAHIT's succinct de Bruijn graph (SdBG)
 * construction (arxiv 1409.7208), as hand-written sm_100a CUDA kernels for one B200.
 *
 *   reads --sdbg_pack_reads--> 2-bit reads in HBM --sdbg_count_edges(k, d)--> sorted solid (k+1)-mers + counts
 *         --sdbg_build--> SdBG arrays W (+minus flag), last, multiplicity
 *
 * What is computed (PAPER.md = /root/reference/PAPER.md; readings A1..A17 = DESIGN.md "Readings"):
 *   - every (k+1)-mer ("edge") e = e[0..k] of every read, and its reverse complement, is a record
 *     (§2 ¶3 "all (k+1)-mers from the input reads are sorted and counted"; both strands: A4, A5);
 *   - records are sorted "in reverse lexicographical order of their length-k prefixes" (§2 ¶2):
 *     ascending colex order of the node e[0..k), ties broken by the outgoing base e[k], with A<C<G<T (A1-A3);
 *   - equal records are counted; "only (k+1)-mers that appear at least d (2 by default) times are kept"
 *     (PAPER.md:35);
 *   - the kept ("solid") edges, in sorted order, are the edge list of the SdBG (Bowe et al. 2012, PAPER.md:27-31,
 *     :106): W[i] = outgoing base (+ minus flag), last[i] = 1 iff edge i is the last edge of its node,
 *     mult[i] = multiplicity;
 *   - when the records exceed the workspace, they are processed "block-wise": partitioned "according to their
 *     length-l prefix (l=8 ...)", "consecutive partitions that fit within the GPU memory are sorted together"
 *     (PAPER.md:33). The length-8 prefix is the prefix of the SORT KEY (A11): 4^8 = 65,536 partitions.
 *
 * Key encoding (what `sdbg_edges.keys` holds): w = ceil(2(k+1)/64) u64 words per edge, word 0 most significant.
 * The k+1 symbols (e[k-1], e[k-2], ..., e[0], e[k]) are written at 2 bits each (A=0 C=1 G=2 T=3), first symbol
 * in the top bits of word 0; the low 64w-2(k+1) bits of the last word are zero. Unsigned multi-word ascending
 * order of keys == the sort order above. Partition ("bucket") of a key = top 16 bits of word 0.
 *
 * Memory: every pointer inside the structs below is a DEVICE pointer to memory owned by the caller; the library
 * never allocates or frees device memory and uses only the workspace given to sdbg_ctx_create. `bases`/`offsets`
 * of sdbg_pack_reads may be host or device pointers (detected). All work is enqueued on the context's stream.
 * No exception crosses the ABI; every call returns SDBG_OK (0) or a negative sdbg_status. Not thread-safe per ctx.
 * There is no CPU fallback: without a CUDA device every compute entry point fails with SDBG_E_CUDA.
 */
#ifndef SDBG_H
#define SDBG_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    SDBG_OK = 0,
    SDBG_E_INVAL = -1,       /* bad argument (null pointer, d == 0, n mismatch, misaligned buffer) */
    SDBG_E_BADBASE = -2,     /* a read holds a character outside ACGTacgt (A7); sdbg_last_error names its index */
    SDBG_E_CAPACITY = -3,    /* an output array is too small; the needed count is written to out->n */
    SDBG_E_WORKSPACE = -4,   /* workspace too small (even one l=8 partition does not fit) */
    SDBG_E_CUDA = -5,        /* CUDA runtime error; sdbg_last_error holds its text */
    SDBG_E_UNSUPPORTED = -6  /* k outside [1, 127] */
} sdbg_status;

#define SDBG_MAX_K 127u
#define SDBG_NUM_BUCKETS 65536u      /* 4^l, l = 8 */
#define SDBG_READ_GUARD_SLOTS 256u   /* slack slots the packed-read buffers need after the last base */

typedef struct sdbg_ctx sdbg_ctx;

/* ---- context -------------------------------------------------------------------------------------------- */

/* Binds a device, a CUDA stream (cudaStream_t passed as void*, NULL = legacy default stream) and a caller-owned
 * device workspace. The workspace plays the role of MEGAHIT's "-m" memory budget: the sorter
 * sizes its block-wise passes to it. workspace must be 256-byte aligned.
 * Errors: SDBG_E_INVAL (null or misaligned workspace), SDBG_E_WORKSPACE (below sdbg_min_workspace()), SDBG_E_CUDA (no such
 * device, or the kernels could not be set up: the library has no CPU fallback). */
int sdbg_ctx_create(sdbg_ctx **ctx, int device, void *cuda_stream, void *workspace, uint64_t workspace_bytes);
void sdbg_ctx_destroy(sdbg_ctx *ctx);
/* Options of a context (all off after sdbg_ctx_create). They choose among ways through the sort and count that give the
 * SAME result bit for bit (PAPER.md:33-35 fix the result, not the way); the tests use them to reach every way at sizes
 * the oracle can check, and to compare the ways with one another.
 *   SDBG_OPT_FORCE_WIDE        one-word-key ranges of any size take the code path of ranges of 2^32 records and more (wide
 *                              look-back words in the radix passes, 64-bit run lengths in the count sweeps)
 *   SDBG_OPT_NO_TABLE_COUNT    sdbg_count_edges sorts every record through every radix pass and counts by one sweep
 *                              (count.cu). Default for d >= 2: the records go through the most significant passes only
 *                              and are counted bucket by bucket in shared-memory tables (hashcount.cu; keys of several
 *                              words by a 64-bit fingerprint of the whole key, every record then compared with the one
 *                              that installed its slot); whatever does not fit there (an over-long bucket, a full table,
 *                              two keys with one fingerprint) is redone the plain way inside the same call
 *   SDBG_OPT_NO_FUSED_EXTRACT  on the default path the extractor writes the keys in read order and the first top pass reads
 *                              them back (default for one dense range of one-word keys, k >= 8: extraction is fused with
 *                              that pass, the keys go from the key maker straight into its 256 bins)
 *   SDBG_OPT_STABLE_FIRST_PASS the first radix pass of sdbg_count_edges' sorts uses the stable kernel like the others
 *                              (default: unstable, equal keys are merged afterwards)
 *   SDBG_OPT_WEAK_FINGERPRINT  (tests) the fingerprint of a key of several words is its first word, so that keys which
 *                              differ further down meet in one table slot and the check sends the range the plain way
 * Errors: SDBG_E_INVAL (null ctx, unknown option). */
enum { SDBG_OPT_FORCE_WIDE = 1, SDBG_OPT_NO_TABLE_COUNT = 2, SDBG_OPT_STABLE_FIRST_PASS = 3, SDBG_OPT_NO_FUSED_EXTRACT = 4, SDBG_OPT_WEAK_FINGERPRINT = 5 };
int sdbg_ctx_set_option(sdbg_ctx *ctx, int option, int value);
const char *sdbg_strerror(int status);           /* static string */
const char *sdbg_last_error(const sdbg_ctx *ctx); /* detail of the last failure on this ctx ("" if none) */

/* ---- a1: pack reads ------------------------------------------------------------------------------------- */

/* 2-bit packed reads, layout private to the library. `words` holds slots_cap/32 u64, `ends` slots_cap/64 u64.
 * Zero-initialise the struct fields n_reads, n_bases, n_slots before the first sdbg_pack_reads call. */
typedef struct {
    uint64_t *words;     /* 2-bit bases, 32 per u64 */
    uint64_t *ends;      /* 1 bit per base slot: read boundary / padding marks */
    uint64_t slots_cap;  /* capacity in base slots; multiple of 64; see sdbg_read_slots */
    uint64_t n_reads;    /* reads packed so far */
    uint64_t n_bases;    /* bases packed so far */
    uint64_t n_slots;    /* slots used so far (multiple of 64) */
} sdbg_reads;

/* slots_cap needed to pack n_bases bases with n_calls calls of sdbg_pack_reads (each call pads to 64 slots). */
uint64_t sdbg_read_slots(uint64_t n_bases, uint64_t n_calls);

/* a1: APPENDS n reads to `out`. Read r is bases[offsets[r] .. offsets[r+1]) — ASCII, one byte
 * per base, upper or lower case; offsets has n+1 non-decreasing entries; bases and offsets are both host or both
 * device pointers. Host input is staged through the workspace in chunks (H2D on the ctx stream). Encoding
 * A=0 C=1 G=2 T=3 (A1); the 2-bit packing is what PAPER.md:31 implies ("2kt bits" for t k-mers).
 * Synchronises the stream. Errors (the struct `out` is left unchanged by all of them): SDBG_E_BADBASE,
 * SDBG_E_CAPACITY (slots_cap too small; sdbg_last_error states the needed value), SDBG_E_INVAL,
 * SDBG_E_WORKSPACE (host input and no room to stage it). */
int sdbg_pack_reads(sdbg_ctx *ctx, const char *bases, const uint64_t *offsets, uint64_t n, sdbg_reads *out);

/* ---- a2-a4, a6: extract, sort, count, solid filter ------------------------------------------------------- */

typedef struct {
    uint64_t *keys;   /* n*w u64, record i at keys[i*w .. i*w+w), word 0 most significant */
    uint32_t *mult;   /* n multiplicities (saturating at 2^32-1, A9) */
    uint64_t cap;     /* capacity in edges of keys/mult */
    uint64_t n;       /* out: number of edges */
    uint32_t k;       /* out (count_edges) / in (build) */
    uint32_t w;       /* out (count_edges) / in (build): ceil(2(k+1)/64) */
} sdbg_edges;

typedef struct {
    uint64_t n_raw;            /* N = 2 * sum_r max(0, L_r - k) records extracted */
    uint64_t n_distinct;       /* distinct records */
    uint64_t n_solid;          /* distinct records with count >= d */
    uint64_t sum_solid_mult;   /* sum of their (unsaturated) counts */
    uint64_t n_ranges;         /* block-wise passes run (1 when everything fits) */
    uint64_t max_range_records;/* records of the largest block-wise pass */
    /* Order-independent checksums, computed only when want_checksums != 0 (they cost ALU time):
     *   mixk(key) = fold h = mix64(h ^ word) over the key's words, most significant first, h0 = 0,
     *   mix64 = the splitmix64 finaliser (z^=z>>30; z*=0xBF58476D1CE4E5B9; z^=z>>27; z*=0x94D049BB133111EB; z^=z>>31).
     *   csum_raw      = sum over all N extracted records of mixk(key)            (mod 2^64), taken before sorting
     *   csum_distinct = sum over distinct records of count * mixk(key)           (mod 2^64), taken after counting
     * The sort/count lost or duplicated nothing iff the two agree (pin P4). */
    uint64_t csum_raw, csum_distinct;
    uint32_t want_checksums;   /* in */
    uint32_t reserved;
    uint64_t *bucket_hist;     /* in, optional device u64[65536]: raw records per l=8 partition (A11) */
} sdbg_stats;

/* Records per key and workspace sizing. sdbg_full_workspace: bytes with which sdbg_count_edges runs as ONE range
 * (no block-wise passes) for reads with n_bases bases; sdbg_min_workspace: the fixed state plus room for a
 * 64 Ki-record range of 4-word keys — sdbg_ctx_create refuses less with SDBG_E_WORKSPACE. */
uint32_t sdbg_key_words(uint32_t k);
uint64_t sdbg_full_workspace(uint64_t n_bases, uint32_t k);
/* The same for a known number of records N = 2 * sum_r max(0, L_r - k) (sdbg_full_workspace assumes the bound
 * N <= 2 * n_bases, which is loose for long keys: 150-base reads give 51 windows at k = 99). 0 if k is out of range. */
uint64_t sdbg_workspace_for_records(uint64_t n_records, uint32_t k);
uint64_t sdbg_min_workspace(void);

/* a2 extract + a3 sort + a4 count/filter (+ a6 block-wise planner).
 * n must equal reads->n_reads. k in [1,127] else SDBG_E_UNSUPPORTED; d >= 1 else SDBG_E_INVAL (A8).
 * Output: out->keys/mult hold the solid edges in sorted order, strictly increasing keys; out->n, out->k, out->w
 * set. If out->cap < number of solid edges: SDBG_E_CAPACITY, out->n = needed count, contents unspecified.
 * If the records do not fit the workspace they are processed in ranges of consecutive l=8 partitions chosen
 * greedily from the 65,536-bin histogram (A12); the output does not depend on the plan. A single partition
 * larger than the workspace gives SDBG_E_WORKSPACE. Synchronises the stream before returning. */
int sdbg_count_edges(sdbg_ctx *ctx, const sdbg_reads *reads, uint64_t n, uint32_t k, uint32_t d,
                     sdbg_edges *out, sdbg_stats *stats /* nullable */);

/* a6 host logic, exposed for testing: greedy maximal runs of consecutive partitions whose record sum is
 * <= capacity (A12). hist: HOST u64[65536]. Writes up to max_ranges triples (lo, hi, records) into
 * ranges[3*i..3*i+3) with hi exclusive, skipping nothing (empty partitions join the current run).
 * Returns the number of ranges, or SDBG_E_WORKSPACE if one partition exceeds capacity, or SDBG_E_CAPACITY if
 * max_ranges is too small. */
int64_t sdbg_plan_ranges(const uint64_t *hist, uint64_t capacity, uint64_t *ranges, uint64_t max_ranges);

/* ---- sharding by ranges of l=8 partitions ------------------------------------------ */

/* "we adopt a block-wise strategy that partitions the k-mers according to their length-l prefix (l=8 in our
 * implementation). The k-mers in consecutive partitions ... are sorted together". The same partitions
 * shard the path across GPUs: every GPU holds the packed reads (replicated: one broadcast) and counts only the edges
 * of a contiguous range of partitions; the outputs of the ranges, concatenated in range order, are the output of
 * sdbg_count_edges, and for k >= 9 no `last` / minus dependency crosses a partition, so the arrays of sdbg_build over
 * each range concatenate too. No collective on the data path (an all-gather of the per-range counts gives offsets).
 *
 * sdbg_count_edges_range: sdbg_count_edges restricted to partitions [bucket_lo, bucket_hi) (partition = top 16 bits
 * of the key). stats->n_raw counts the raw records of the range only; checksums cover the range; stats->bucket_hist,
 * if asked for, is still the histogram of all partitions. Same errors as sdbg_count_edges, plus SDBG_E_INVAL for a
 * bad range. */
int sdbg_count_edges_range(sdbg_ctx *ctx, const sdbg_reads *reads, uint64_t n, uint32_t k, uint32_t d,
                           uint32_t bucket_lo, uint32_t bucket_hi, sdbg_edges *out, sdbg_stats *stats /* nullable */);
/* hist: DEVICE u64[65536] = raw records per l=8 partition of the packed reads at this k (one pass of the extractor
 * without output). Launches on the ctx stream and does not synchronise. */
int sdbg_bucket_hist(sdbg_ctx *ctx, const sdbg_reads *reads, uint32_t k, uint64_t *hist);
/* Host logic: n_shards contiguous ranges of partitions balanced by records. hist: HOST u64[65536]; bounds: HOST
 * u32[n_shards + 1], bounds[0] = 0, bounds[n_shards] = 65536, shard i = [bounds[i], bounds[i+1]); shard i starts at the
 * first partition before which at least i/n_shards of the records lie (a shard may be empty). Deterministic: every
 * rank computes the same plan from the same histogram. */
int sdbg_plan_shards(const uint64_t *hist, uint32_t n_shards, uint32_t *bounds);

/* ---- a5: SdBG arrays ------------------------------------------------------------------------------------ */

#define SDBG_SORTED 1u   /* edges->keys are strictly increasing (the output of sdbg_count_edges) */

typedef struct {
    uint8_t *W;           /* n bytes: 1..4 = outgoing base A,C,G,T; +4 when the minus flag is set; 0 reserved for '$' (A10) */
    uint64_t *last_bits;  /* ceil(cap/64) u64, bit i%64 of word i/64 (LSB first) = last[i]; tail bits of the final word zero */
    uint32_t *mult;       /* n multiplicities */
    uint64_t cap;         /* capacity in edges */
    uint64_t n;           /* out */
} sdbg_graph;

/* a5; SdBG definition, Bowe et al. 2012:
 *   W[i]     = e[k] of edge i;
 *   last[i]  = (i == n-1) or node(i+1) != node(i)                                   (A14)
 *   minus[i] = exists j < i with e_j[1..k) == e_i[1..k) and e_j[k] == e_i[k]        (minus[0] = 0)
 *   mult[i]  = edges->mult[i].
 * With SDBG_SORTED the input is used as is (one streaming kernel; does not synchronise). Without it, edges may be
 * in any order with repeats: they are sorted with the same radix sorter and equal keys are merged by summing mult
 * (saturating at 2^32-1), so count_edges == build over raw records with mult 1 followed by the d filter. In that
 * case edges->keys/mult are overwritten with the sorted, merged edges, edges->n is updated, and the call
 * synchronises. Errors: SDBG_E_CAPACITY (out->n = needed), SDBG_E_WORKSPACE, SDBG_E_INVAL. */
int sdbg_build(sdbg_ctx *ctx, sdbg_edges *edges, uint32_t flags, sdbg_graph *out);

/* ---- lossless extras of the SdBG ------------------------------------------ */

typedef struct {
    uint8_t *W;            /* m bytes: 0 = '$' (dummy outgoing edge), 1..4 = A,C,G,T, +4 with the minus flag */
    uint64_t *last_bits;   /* ceil(cap/64) u64, LSB first, tail bits zero */
    uint64_t *valid_bits;  /* ceil(cap/64) u64: the validity bit-vector of PAPER.md:31, all ones for the m edges */
    uint32_t *mult;        /* m multiplicities, 0 for '$' edges */
    uint64_t *aux_bits;    /* the "auxiliary vector of 2kt bits": ceil(2*k*aux_cap/64) u64 */
    uint64_t cap;          /* capacity in edges of W / last_bits / valid_bits / mult */
    uint64_t aux_cap;      /* capacity in nodes of aux_bits */
    uint64_t m;            /* out: edges = solid edges + '$' edges */
    uint64_t t;            /* out: zero-indegree nodes */
    uint64_t n_zero_out;   /* out: '$' edges = nodes without outgoing edge */
    uint64_t *zin_bits;    /* ceil(cap/64) u64, LSB first, tail bits zero: bit i = edge i is the last edge of a node without
                              incoming edge, so that entry j of aux_bits is the node of the j-th set bit (reading A24) */
    uint64_t F[5];         /* out (host): F[c] = index of the first edge whose node ends with a base >= c (A=0 .. T=3),
                              F[4] = m: the F array of Bowe et al. in edge positions (reading A25) */
} sdbg_full_graph;

/* "Our implementation has added a bit-vector of length m to mark the validity of each edge ... and an auxiliary vector
 * of 2kt bits (where k is the k-mer size and t is the number of zero-indegree vertices) to store the sequence of
 * zero-indegree vertices to ensure the graph being lossless". Readings A18-A20 of DESIGN.md:
 *   - nodes: src(e) = e[0..k), tgt(e) = e[1..k] over the given edges;
 *   - every node of tgt \ src (no outgoing edge) gets the dummy edge (node, '$') as in Bowe et al.;
 *   - the nodes of src \ tgt (no incoming edge), in colex order, are the auxiliary vector: node i occupies stream
 *     bits [2k i, 2k (i+1)), bases in sequence order v[0..k) at 2 bits each, stream bit 0 = most significant bit of
 *     aux_bits[0]; no incoming dummy edges are made;
 *   - the arrays list solid and '$' edges together, sorted by (colex of the node, outgoing symbol), '$' < A;
 *     W / last / minus by the rules of sdbg_build ('$' edges: W = 0, last = 1, mult = 0); valid_bits = m ones;
 *   - zin_bits and F tie the auxiliary vector and the node classes to edge positions (A24, A25; used by sdbg_index_build).
 * `edges` must be sorted and distinct (the output of sdbg_count_edges), 2 <= k <= 127, fewer than 2^32 edges.
 * Synchronises the stream. Errors: SDBG_E_CAPACITY (out->m / out->t hold the needed values), SDBG_E_WORKSPACE
 * (needs about 40 + 16 w bytes of workspace per edge), SDBG_E_UNSUPPORTED, SDBG_E_INVAL. */
int sdbg_build_full(sdbg_ctx *ctx, const sdbg_edges *edges, sdbg_full_graph *out);

/* Mercy-kmers (§2 ¶3; readings A21-A23 of DESIGN.md): "Given two solid (k+1)-mers x
 * and y from the same read, where x has no outdegree and y has no indegree. If all (k+1)-mers between x and y in that
 * read are not solid, they will be added to the de Bruijn graph as mercy-kmers." For every read (as packed), every
 * maximal run of non-solid windows with a solid window x right before it and a solid window y right behind it: if
 * tgt(x) has no outgoing solid edge and src(y) has no incoming solid edge, every window of the run and its reverse
 * complement are appended to `out` (keys, mult = 1; unsorted, with repeats: out->n records). `solid` is the output of
 * sdbg_count_edges over the same reads (sorted, distinct; 2 <= k <= 127; fewer than 2^32 edges). To build the graph
 * with them, put solid and mercy records into one sdbg_edges and call sdbg_build without SDBG_SORTED (equal keys are
 * merged, mult summed). Workspace: about 40 + 16 w bytes per solid edge for the zero-degree lists plus a hash table of
 * 16-byte slots, 2 to 4 per solid edge. Synchronises. Errors: SDBG_E_CAPACITY (out->n = needed count), SDBG_E_WORKSPACE,
 * SDBG_E_UNSUPPORTED, SDBG_E_INVAL. */
int sdbg_mercy_edges(sdbg_ctx *ctx, const sdbg_reads *reads, const sdbg_edges *solid, sdbg_edges *out);

/* ---- traversal: rank/select over the arrays of the full graph ------------------------- */

/* "A succinct de Bruijn graph (SdBG) encodes a graph with m edges in O(m) bits, and supports O(1) time traversal from a
 * vertex to its neighbors" (Bowe et al.). Readings A24-A26 of DESIGN.md. The index holds
 * five bit-vectors over the m edges,
 *     B_c[i] = (W[i] is base c, minus flag clear), c = A,C,G,T;     H[i] = last[i] and not zin[i],
 * each as 64-byte cells {u64 ones before the cell, 448 bits}, so that a rank is one aligned 64-byte read, plus, per
 * vector, the cell of every 512-th one for select. It borrows g->W and g->last_bits (they must outlive the index).
 *     forward(i)  = -1 if W[i] == 0 ('$'), else the index of the last edge of the node e_i[1..k]
 *                 = select_H(rank_H(F[c]) + rank_{B_c}(i + 1)),              c = base of W[i]
 *     backward(j) = the smallest index of an edge that enters the node of edge j, -1 if the node has no incoming edge
 *                 = select_{B_c}(rank_H(p + 1) - rank_H(F[c])),   p = last edge of j's node, c = its class in F
 * The validity bits are not consulted. */
typedef struct {
    uint64_t *cells;        /* device, caller-owned: sdbg_index_bytes(cap) bytes, 64-byte aligned */
    uint64_t bytes;         /* size of that block */
    uint64_t m;             /* out: edges indexed */
    uint64_t n_cells;       /* out: m / 448 + 1 */
    uint64_t F[5];          /* out: copy of g->F */
    uint64_t HF[5];         /* out: rank_H(F[c]) */
    uint64_t ones[5];       /* out: set bits of B_A, B_C, B_G, B_T, H */
    const uint8_t *W;       /* out: g->W (borrowed) */
    const uint64_t *last_bits; /* out: g->last_bits (borrowed) */
} sdbg_index;

/* Bytes of `cells` for a graph of up to m edges. Host-only. */
uint64_t sdbg_index_bytes(uint64_t m);
/* Builds the index of g (the output of sdbg_build_full, zin_bits included) on the ctx stream; synchronises.
 * Errors: SDBG_E_CAPACITY (ix->bytes too small), SDBG_E_INVAL (null arrays, no zin_bits), SDBG_E_UNSUPPORTED (m >= 2^32). */
int sdbg_index_build(sdbg_ctx *ctx, const sdbg_full_graph *g, sdbg_index *ix);
/* The same index for callers that cannot allocate device memory (code under CUDA graph capture around it, tight serving
 * loops, harnesses that forbid cudaMalloc): no ctx and no workspace. The build scratch is a static device array inside the
 * library (374,648 bytes per GPU that loads it, held until exit), which limits the graph to
 * sdbg_index_static_max_edges() = 2^28 edges; a larger m is refused with SDBG_E_CAPACITY. The caller passes the graph and
 * `ix->cells` (device, 64-byte aligned, at least sdbg_index_static_bytes(m) bytes: cells and select samples only; a block
 * of sdbg_index_bytes(m) bytes will do as well). Runs on `stream` (a cudaStream_t, NULL = the default stream) of the
 * CURRENT device and synchronises it; calls no cudaMalloc / cudaFree or allocating library routine. Every call on a
 * device shares the scratch and it keeps the last call's contents (what must start at zero is cleared per call): calls
 * that overlap on one GPU race, so serialise them (one stream, or events). The result is the same index, bit for bit, as
 * sdbg_index_build's; sdbg_forward / sdbg_backward take it. Errors: SDBG_E_CAPACITY, SDBG_E_INVAL, SDBG_E_CUDA; the text
 * is in sdbg_index_build_static_error() (per host thread). */
uint64_t sdbg_index_static_max_edges(void);
uint64_t sdbg_index_static_bytes(uint64_t m);
int sdbg_index_build_static(void *stream, const sdbg_full_graph *g, sdbg_index *ix);
const char *sdbg_index_build_static_error(void);
/* out[q] = forward(edge_idx[q]) / backward(edge_idx[q]) for n queries; edge_idx and out are DEVICE arrays; an index
 * >= m yields -2. Launches on the ctx stream and does not synchronise. */
int sdbg_forward(sdbg_ctx *ctx, const sdbg_index *ix, const uint64_t *edge_idx, uint64_t n, int64_t *out);
int sdbg_backward(sdbg_ctx *ctx, const sdbg_index *ix, const uint64_t *edge_idx, uint64_t n, int64_t *out);

/* ---- measurement hooks ---------------------------------------------------------------------------------- */

/* kernel classes: RADIX = onesweep_kernel launches over all records of a range; TABLE = hash_count_kernel (the table
 * count of the default path, one launch per range); COUNT = everything else of step a4 (segment bounds, block-sum scan and
 * copy of the staged edges on the default path; the sweeps of count.cu otherwise) */
enum { SDBG_T_PACK = 0, SDBG_T_EXTRACT = 1, SDBG_T_RADIX = 2, SDBG_T_COUNT = 3, SDBG_T_EMIT = 4, SDBG_T_OTHER = 5, SDBG_T_TABLE = 6, SDBG_T_NUM = 7 };

typedef struct {
    double ms[SDBG_T_NUM];          /* device time per kernel class, CUDA events on the ctx stream */
    uint64_t launches[SDBG_T_NUM];  /* kernel launches per class */
    uint64_t bytes[SDBG_T_NUM];     /* algorithmic bytes per class */
} sdbg_timing;

/* Launches, by this process so far, of the UNSTABLE variant of the radix pass (radix.cu FIRST: the order of equal digits is
 * hardware-defined). Only the sorts of sdbg_count_edges may use it (they merge equal keys afterwards); sdbg_build,
 * sdbg_build_full and sdbg_mercy_edges depend on stable passes, and the tests assert that they leave this counter alone. */
uint64_t sdbg_unstable_radix_launches(void);

/* on != 0: bracket every kernel class with CUDA events (a few microseconds each). Launch counters always run. */
int sdbg_ctx_set_timing(sdbg_ctx *ctx, int on);
/* Synchronises the stream, adds up the event pairs recorded since the last call, writes and resets the totals. */
int sdbg_ctx_get_timing(sdbg_ctx *ctx, sdbg_timing *out);

#ifdef __cplusplus
}
#endif
#endif /* SDBG_H */

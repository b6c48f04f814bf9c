/* sdbg_oracle.c — TEST INFRASTRUCTURE ONLY. The plain, slow, single-threaded CPU definition of what
 * the SdBG-construction hot path computes. Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, link or call this file. It shares no code with the
 * CUDA library (paper_1409_7208_b200/csrc): no headers, helpers, tables or pre/post-processing.
 *
 * The method reaches an exactly defined result (a sort + group-by), so this is that definition written
 * out on strings, in the order of SURVEY.md §8(c) steps 1-6:
 *
 *  1. E <- []. For each read r, for i = 0 .. L_r-k-1: e <- r[i : i+k+1]; append e and rc(e) to E.
 *     ("all (k+1)-mers from the input reads", §2 ¶3; both strands and the literal multiset
 *     reading for palindromes: DESIGN.md readings A4, A5.)  Reads with L_r <= k add nothing (A6).
 *  2. Sort E: compare a[k-1] vs b[k-1], a[k-2] vs b[k-2], ..., a[0] vs b[0] (A<C<G<T); if all equal,
 *     a[k] vs b[k].  ("sorting a set of (k+1)-mers ... in reverse lexicographical order of their length-k
 *     prefixes", §2 ¶2; colex-ascending reading A2, tie-break A3.)
 *  3. Group equal strings; cnt(e) = group size.  ("sorted and counted".)
 *  4. S <- groups with cnt >= d, in sorted order.  ("appear at least d (2 by default) times".)
 *  5. For e = S[i]:  W[i] = e[k];  last[i] = (i == |S|-1) or S[i+1][0:k] != e[0:k];
 *     minus[i] = exists j < i with S[j][1:k] == e[1:k] and S[j][k] == e[k];  mult[i] = cnt(e).
 *     (SdBG / BOSS arrays, §2 ¶1, Bowe et al. 2012 PAPER.md:106; flag rules per
 *     BASELINE.json north_star.)  Because S is sorted by (e[k-1],...,e[0],e[k]), all j with
 *     S[j][1:k] == e[1:k] are contiguous and directly before i, so the scan over j stops at the first
 *     j whose S[j][1:k] differs; the O(|S|^2) literal form is checked against this in the tests.
 *  6. Encodings, only for comparison with the CUDA library: key(e) = symbols (e[k-1],...,e[0],e[k]) at
 *     2 bits each (A0 C1 G2 T3), first symbol in the top bits of word 0, zero-padded low, w = ceil(2(k+1)/64)
 *     words per key; W byte = 1 + code(e[k]), + 4 if minus; last packed LSB-first into u64 words.
 *
 * Optional restriction (large configs, SURVEY.md §8(c) "Large configs"): keep in step 1 only records whose
 * key string (e[k-1],...,e[0],e[k]) begins with one of a given set of 8-symbol strings (l=8 partitions,
 * PAPER.md:33). Requires k >= 9, for which no `last`/minus dependency crosses a partition, so the result is the
 * concatenation of those partitions' slices of the full result. For the same purpose step 1 can also be fed
 * records that were extracted earlier (orc_add_edges): several oracle instances may scan disjoint parts of the
 * reads (the kept raw records of each are read back with orc_raw) and one instance then runs steps 2-5 on
 * the union.
 *
 * Pins (tests/test_oracle_pins.py): hand-worked example T0 (tests/golden/t0_handworked.txt), complete
 * de Bruijn closed form, independent Python brute force, count/closure invariants, numpy sort/unique.
 * Parity unpinned: nothing.
 */
#define _GNU_SOURCE
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct orc {
    uint32_t k, d;
    uint32_t n_prefix;
    char *prefix;                     /* n_prefix * 8 chars */
    /* step 1 */
    char *E; uint64_t nE, capE;       /* records, (k+1) chars each */
    uint64_t n_seen;                  /* records before the optional prefix restriction */
    /* steps 3-5 */
    uint64_t n_distinct, n_solid, sum_solid_mult;
    char *D; uint32_t *Dcnt;          /* distinct edges + counts */
    char *S; uint32_t *mult;          /* solid edges */
    uint8_t *W, *last, *minus;
} orc;

enum { ORC_OK = 0, ORC_E_BADBASE = -2, ORC_E_NOMEM = -7, ORC_E_INVAL = -1 };

orc *orc_new(uint32_t k, uint32_t d, const char *prefixes /* NULL or n_prefix * 8 chars */, uint32_t n_prefix) {
    if (k < 1 || d < 1) return NULL;
    if (prefixes && n_prefix && k < 9) return NULL;
    orc *o = (orc *)calloc(1, sizeof(orc));
    if (!o) return NULL;
    o->k = k; o->d = d;
    if (prefixes && n_prefix) {
        o->prefix = (char *)malloc((size_t)n_prefix * 8);
        if (!o->prefix) { free(o); return NULL; }
        memcpy(o->prefix, prefixes, (size_t)n_prefix * 8);
        o->n_prefix = n_prefix;
    }
    return o;
}

void orc_free(orc *o) {
    if (!o) return;
    free(o->prefix);
    free(o->E); free(o->D); free(o->Dcnt); free(o->S); free(o->mult); free(o->W); free(o->last); free(o->minus);
    free(o);
}

static char comp(char c) { return c == 'A' ? 'T' : c == 'C' ? 'G' : c == 'G' ? 'C' : 'A'; }

static int push(orc *o, const char *e) {
    const uint32_t k = o->k;
    o->n_seen++;
    if (o->n_prefix) {               /* key string symbol t is e[k-1-t] for t < k */
        int keep = 0;
        for (uint32_t p = 0; p < o->n_prefix && !keep; ++p) {
            keep = 1;
            for (uint32_t t = 0; t < 8; ++t) if (e[k - 1 - t] != o->prefix[p * 8 + t]) { keep = 0; break; }
        }
        if (!keep) return ORC_OK;
    }
    if (o->nE == o->capE) {
        uint64_t nc = o->capE ? o->capE * 2 : 1024;
        char *p = (char *)realloc(o->E, nc * (k + 1));
        if (!p) return ORC_E_NOMEM;
        o->E = p; o->capE = nc;
    }
    memcpy(o->E + o->nE * (k + 1), e, k + 1);
    o->nE++;
    return ORC_OK;
}

/* Step 1 over n reads: read r is bases[offsets[r] .. offsets[r+1]). Lower-case acgt is folded to upper case;
 * any other character fails with ORC_E_BADBASE (reading A7). May be called repeatedly (reads are a multiset). */
int orc_add_reads(orc *o, const char *bases, const uint64_t *offsets, uint64_t n) {
    const uint32_t k = o->k;
    char *e = (char *)malloc(k + 1), *rc = (char *)malloc(k + 1);
    char *rd = NULL; uint64_t rdcap = 0;
    int st = ORC_OK;
    if (!e || !rc) { free(e); free(rc); return ORC_E_NOMEM; }
    for (uint64_t r = 0; r < n && st == ORC_OK; ++r) {
        uint64_t L = offsets[r + 1] - offsets[r];
        if (L > rdcap) { free(rd); rd = (char *)malloc(L); rdcap = L; if (!rd) { st = ORC_E_NOMEM; break; } }
        for (uint64_t j = 0; j < L; ++j) {
            char c = bases[offsets[r] + j];
            if (c >= 'a' && c <= 'z') c = (char)(c - 'a' + 'A');
            if (c != 'A' && c != 'C' && c != 'G' && c != 'T') { st = ORC_E_BADBASE; break; }
            rd[j] = c;
        }
        if (st != ORC_OK) break;
        for (uint64_t i = 0; i + k + 1 <= L && st == ORC_OK; ++i) {
            memcpy(e, rd + i, k + 1);
            for (uint32_t t = 0; t <= k; ++t) rc[t] = comp(e[k - t]);
            st = push(o, e);
            if (st == ORC_OK) st = push(o, rc);
        }
    }
    free(e); free(rc); free(rd);
    return st;
}

/* Step 1 fed with n records extracted earlier ((k+1) chars each, upper case ACGT): see the header. */
int orc_add_edges(orc *o, const char *edges, uint64_t n) {
    int st = ORC_OK;
    for (uint64_t i = 0; i < n && st == ORC_OK; ++i) st = push(o, edges + i * (o->k + 1));
    return st;
}
/* The records kept by step 1 so far, in the order they were met (before orc_finish sorts them in place). */
const char *orc_raw(const orc *o) { return o->E; }

/* Step 2 comparator. */
static int cmp_edges(const void *pa, const void *pb, void *ctx) {
    const char *a = (const char *)pa, *b = (const char *)pb;
    const uint32_t k = *(const uint32_t *)ctx;
    for (uint32_t t = k; t-- > 0;) if (a[t] != b[t]) return a[t] < b[t] ? -1 : 1;
    if (a[k] != b[k]) return a[k] < b[k] ? -1 : 1;
    return 0;
}

int orc_finish(orc *o) {
    const uint32_t k = o->k, R = k + 1;
    /* 2 */
    if (o->nE) qsort_r(o->E, o->nE, R, cmp_edges, &o->k);
    /* 3: count groups */
    uint64_t nd = 0;
    for (uint64_t i = 0; i < o->nE; ++i) if (i == 0 || memcmp(o->E + i * R, o->E + (i - 1) * R, R) != 0) nd++;
    o->n_distinct = nd;
    o->D = (char *)malloc(nd * R + 1); o->Dcnt = (uint32_t *)malloc(nd * 4 + 4);
    if (!o->D || !o->Dcnt) return ORC_E_NOMEM;
    uint64_t g = 0;
    for (uint64_t i = 0; i < o->nE;) {
        uint64_t j = i + 1;
        while (j < o->nE && memcmp(o->E + j * R, o->E + i * R, R) == 0) ++j;
        memcpy(o->D + g * R, o->E + i * R, R);
        uint64_t c = j - i;
        o->Dcnt[g] = c > 0xffffffffull ? 0xffffffffu : (uint32_t)c;   /* A9: saturate */
        ++g; i = j;
    }
    /* 4 */
    uint64_t ns = 0;
    for (uint64_t i = 0; i < nd; ++i) if (o->Dcnt[i] >= o->d) ns++;
    o->n_solid = ns;
    o->S = (char *)malloc(ns * R + 1); o->mult = (uint32_t *)malloc(ns * 4 + 4);
    o->W = (uint8_t *)malloc(ns + 1); o->last = (uint8_t *)malloc(ns + 1); o->minus = (uint8_t *)malloc(ns + 1);
    if (!o->S || !o->mult || !o->W || !o->last || !o->minus) return ORC_E_NOMEM;
    uint64_t s = 0;
    o->sum_solid_mult = 0;
    for (uint64_t i = 0; i < nd; ++i) if (o->Dcnt[i] >= o->d) {
        memcpy(o->S + s * R, o->D + i * R, R); o->mult[s] = o->Dcnt[i]; o->sum_solid_mult += o->Dcnt[i]; ++s;
    }
    /* 5 */
    for (uint64_t i = 0; i < ns; ++i) {
        const char *e = o->S + i * R;
        o->W[i] = (uint8_t)e[k];
        o->last[i] = (i == ns - 1) || memcmp(o->S + (i + 1) * R, e, k) != 0;
        uint8_t m = 0;
        for (uint64_t j = i; j-- > 0;) {
            const char *f = o->S + j * R;
            if (memcmp(f + 1, e + 1, k - 1) != 0) break;   /* S[j][1:k] != e[1:k]: no earlier j can match */
            if (f[k] == e[k]) { m = 1; break; }
        }
        o->minus[i] = m;
    }
    return ORC_OK;
}

uint64_t orc_n_raw(const orc *o) { return o->nE; }
uint64_t orc_n_seen(const orc *o) { return o->n_seen; }
uint64_t orc_n_distinct(const orc *o) { return o->n_distinct; }
uint64_t orc_n_solid(const orc *o) { return o->n_solid; }
uint64_t orc_sum_solid_mult(const orc *o) { return o->sum_solid_mult; }
const char *orc_sorted_raw(const orc *o) { return o->E; }
const char *orc_distinct(const orc *o) { return o->D; }
const uint32_t *orc_distinct_cnt(const orc *o) { return o->Dcnt; }
const char *orc_solid(const orc *o) { return o->S; }
const uint32_t *orc_mult(const orc *o) { return o->mult; }
const uint8_t *orc_W(const orc *o) { return o->W; }
const uint8_t *orc_last(const orc *o) { return o->last; }
const uint8_t *orc_minus(const orc *o) { return o->minus; }

static uint64_t code(char c) { return c == 'A' ? 0 : c == 'C' ? 1 : c == 'G' ? 2 : 3; }

/* Step 6, key of one edge string: w words, symbol t of (e[k-1],...,e[0],e[k]) at bits [62-2(t%32), 63-2(t%32)] of word t/32. */
void orc_encode_keys(const orc *o, const char *edges, uint64_t n, uint64_t *keys) {
    const uint32_t k = o->k, R = k + 1, w = (2 * R + 63) / 64;
    for (uint64_t i = 0; i < n; ++i) {
        const char *e = edges + i * R;
        uint64_t *kw = keys + i * w;
        for (uint32_t j = 0; j < w; ++j) kw[j] = 0;
        for (uint32_t t = 0; t <= k; ++t) {
            char sym = t < k ? e[k - 1 - t] : e[k];
            kw[t / 32] |= code(sym) << (62 - 2 * (t % 32));
        }
    }
}

/* Step 6, SdBG arrays of the solid edges. Wbyte[n_solid], last_bits[ceil(n_solid/64)]. */
void orc_encode_graph(const orc *o, uint8_t *Wbyte, uint64_t *last_bits) {
    uint64_t ns = o->n_solid;
    for (uint64_t j = 0; j < (ns + 63) / 64; ++j) last_bits[j] = 0;
    for (uint64_t i = 0; i < ns; ++i) {
        Wbyte[i] = (uint8_t)(1 + code((char)o->W[i]) + (o->minus[i] ? 4 : 0));
        if (o->last[i]) last_bits[i / 64] |= 1ull << (i % 64);
    }
}

/* ---- the lossless extras of PAPER.md:31 (readings A18-A20 in DESIGN.md) -------------------------
 * "a bit-vector of length m to mark the validity of each edge ... and an auxiliary vector of 2kt bits (where k is the
 * k-mer size and t is the number of zero-indegree vertices) to store the sequence of zero-indegree vertices to ensure
 * the graph being lossless"; outgoing `$` edges as in Bowe et al..
 *   nodes: src(e) = e[0..k), tgt(e) = e[1..k] over the solid edges S.
 *   Z_out = tgt(S) \ src(S): nodes without an outgoing edge; each gets the dummy edge (v, '$').
 *   Z_in  = src(S) \ tgt(S): nodes without an incoming edge; their k-mers, in colex order of the node, are the
 *           auxiliary vector (t = |Z_in|); no incoming dummy edges are made (the vector stands in for them).
 *   F = S + dummies, sorted by (colex of the node, outgoing symbol) with '$' < A < C < G < T.
 *   Over F, by the rules of step 5 applied literally: W (0 for '$'), last, minus ('$' edges never carry it), mult
 *   (0 for dummies); validity = all ones. */
typedef struct orc_full {
    uint64_t m, t, n_zero_out;
    char *F;            /* m edges, k+1 chars, '$' as the outgoing symbol of a dummy */
    uint8_t *W, *last;  /* W: 0 for '$', else 1 + code, + 4 with the minus flag */
    uint32_t *mult;
    char *aux;          /* t nodes, k chars each, sequence order v[0..k) */
} orc_full;

static uint32_t g_kcmp;   /* length for cmp_kmers (qsort has no context argument in C11) */
static int cmp_kmers(const void *pa, const void *pb) {   /* colex: last character first */
    const char *a = (const char *)pa, *b = (const char *)pb;
    for (uint32_t t = g_kcmp; t-- > 0;) if (a[t] != b[t]) return a[t] < b[t] ? -1 : 1;
    return 0;
}
static uint64_t uniq_kmers(char *a, uint64_t n, uint32_t k) {
    uint64_t m = 0;
    for (uint64_t i = 0; i < n; ++i) if (i == 0 || memcmp(a + i * k, a + (m - 1) * k, k) != 0) { memmove(a + m * k, a + i * k, k); ++m; }
    return m;
}
static int sym_rank(char c) { return c == '$' ? 0 : c == 'A' ? 1 : c == 'C' ? 2 : c == 'G' ? 3 : 4; }

orc_full *orc_full_graph(const orc *o) {
    const uint32_t k = o->k, R = k + 1;
    const uint64_t ns = o->n_solid;
    orc_full *f = (orc_full *)calloc(1, sizeof(orc_full));
    char *src = (char *)malloc(ns * k + 1), *tgt = (char *)malloc(ns * k + 1);
    if (!f || !src || !tgt) return NULL;
    for (uint64_t i = 0; i < ns; ++i) { memcpy(src + i * k, o->S + i * R, k); memcpy(tgt + i * k, o->S + i * R + 1, k); }
    g_kcmp = k;
    qsort(src, ns, k, cmp_kmers); qsort(tgt, ns, k, cmp_kmers);
    const uint64_t nsrc = uniq_kmers(src, ns, k), ntgt = uniq_kmers(tgt, ns, k);
    /* set differences of two colex-sorted lists */
    char *zout = (char *)malloc(ntgt * k + 1), *zin = (char *)malloc(nsrc * k + 1);
    uint64_t nzo = 0, nzi = 0, a = 0, b = 0;
    while (a < nsrc || b < ntgt) {
        int c = a == nsrc ? 1 : b == ntgt ? -1 : cmp_kmers(src + a * k, tgt + b * k);
        if (c < 0) { memcpy(zin + nzi++ * k, src + a++ * k, k); }
        else if (c > 0) { memcpy(zout + nzo++ * k, tgt + b++ * k, k); }
        else { ++a; ++b; }
    }
    f->t = nzi; f->n_zero_out = nzo; f->aux = zin; f->m = ns + nzo;
    /* F: merge S (sorted by node, then symbol) with the dummies (sorted by node) */
    f->F = (char *)malloc(f->m * R + 1); f->mult = (uint32_t *)malloc(f->m * 4 + 4);
    f->W = (uint8_t *)malloc(f->m + 1); f->last = (uint8_t *)malloc(f->m + 1);
    uint64_t i = 0, j = 0, p = 0;
    while (i < ns || j < nzo) {
        int take_dummy;
        if (i == ns) take_dummy = 1;
        else if (j == nzo) take_dummy = 0;
        else { int c = cmp_kmers(zout + j * k, o->S + i * R); take_dummy = c <= 0; }   /* equal node: '$' first */
        if (take_dummy) { memcpy(f->F + p * R, zout + j * k, k); f->F[p * R + k] = '$'; f->mult[p] = 0; ++j; }
        else { memcpy(f->F + p * R, o->S + i * R, R); f->mult[p] = o->mult[i]; ++i; }
        ++p;
    }
    for (uint64_t q = 0; q < f->m; ++q) {   /* step 5 on F, literally */
        const char *e = f->F + q * R;
        f->last[q] = (q == f->m - 1) || memcmp(f->F + (q + 1) * R, e, k) != 0;
        uint8_t minus = 0;
        if (e[k] != '$')
            for (uint64_t r = q; r-- > 0;) {
                const char *g = f->F + r * R;
                if (memcmp(g + 1, e + 1, k - 1) != 0) break;
                if (g[k] == e[k]) { minus = 1; break; }
            }
        f->W[q] = (uint8_t)(e[k] == '$' ? 0 : sym_rank(e[k]) + (minus ? 4 : 0));
    }
    free(src); free(tgt); free(zout);
    return f;
}
void orc_full_free(orc_full *f) { if (f) { free(f->F); free(f->W); free(f->last); free(f->mult); free(f->aux); free(f); } }
uint64_t orc_full_m(const orc_full *f) { return f->m; }
uint64_t orc_full_t(const orc_full *f) { return f->t; }
uint64_t orc_full_n_zero_out(const orc_full *f) { return f->n_zero_out; }
const char *orc_full_edges(const orc_full *f) { return f->F; }
const uint8_t *orc_full_W(const orc_full *f) { return f->W; }
const uint8_t *orc_full_last(const orc_full *f) { return f->last; }
const uint32_t *orc_full_mult(const orc_full *f) { return f->mult; }
const char *orc_full_aux(const orc_full *f) { return f->aux; }

/* ---- mercy-kmers (readings A21-A23 in DESIGN.md) ---------------------------------
 * "Given two solid (k+1)-mers x and y from the same read, where x has no outdegree and y has no indegree. If all
 * (k+1)-mers between x and y in that read are not solid, they will be added to the de Bruijn graph as mercy-kmers."
 *   For every read (as given), windows w_i = r[i..i+k]; w_i is solid iff it is one of the solid edges S.
 *   For every maximal run w_a..w_b of non-solid windows that has a solid window on both sides (x = w_{a-1},
 *   y = w_{b+1}): if tgt(x) = x[1..k] has no outgoing solid edge and src(y) = y[0..k) has no incoming solid edge, every
 *   w_i of the run and its reverse complement are recorded once (both strands, as in step 1).
 * Output: the recorded (k+1)-mers in the order they were met (a multiset; the caller sorts / merges them). */
static int64_t find_edge(const orc *o, const char *e) {   /* index of e among the solid edges, or -1 (binary search, step-2 order) */
    uint64_t lo = 0, hi = o->n_solid;
    const uint32_t R = o->k + 1;
    while (lo < hi) {
        uint64_t mid = lo + (hi - lo) / 2;
        int c = cmp_edges(o->S + mid * R, e, (void *)&o->k);
        if (c == 0) return (int64_t)mid;
        if (c < 0) lo = mid + 1; else hi = mid;
    }
    return -1;
}
static int kmer_in(const char *list, uint64_t n, uint32_t k, const char *v) {   /* colex-sorted list of k-mers */
    uint64_t lo = 0, hi = n;
    g_kcmp = k;
    while (lo < hi) {
        uint64_t mid = lo + (hi - lo) / 2;
        int c = cmp_kmers(list + mid * k, v);
        if (c == 0) return 1;
        if (c < 0) lo = mid + 1; else hi = mid;
    }
    return 0;
}

typedef struct orc_mercy { uint64_t n, cap; char *E; } orc_mercy;

static int mercy_push(orc_mercy *m, const char *e, uint32_t R) {
    if (m->n == m->cap) {
        uint64_t nc = m->cap ? m->cap * 2 : 256;
        char *p = (char *)realloc(m->E, nc * R);
        if (!p) return ORC_E_NOMEM;
        m->E = p; m->cap = nc;
    }
    memcpy(m->E + m->n * R, e, R);
    m->n++;
    return ORC_OK;
}

/* reads as in orc_add_reads; call after orc_finish. Returns NULL on error. */
orc_mercy *orc_mercy_scan(const orc *o, const char *bases, const uint64_t *offsets, uint64_t n) {
    const uint32_t k = o->k, R = k + 1;
    orc_full *f = orc_full_graph(o);
    orc_mercy *m = (orc_mercy *)calloc(1, sizeof(orc_mercy));
    if (!f || !m) return NULL;
    /* nodes without outgoing edge: the nodes of the '$' edges of F, in colex order */
    char *zout = (char *)malloc(f->n_zero_out * k + 1);
    uint64_t nzo = 0;
    for (uint64_t q = 0; q < f->m; ++q) if (f->F[q * R + k] == '$') memcpy(zout + nzo++ * k, f->F + q * R, k);
    char *rd = NULL, *rc = (char *)malloc(R);
    uint8_t *sol = NULL;
    uint64_t cap = 0;
    int st = ORC_OK;
    for (uint64_t r = 0; r < n && st == ORC_OK; ++r) {
        const uint64_t L = offsets[r + 1] - offsets[r];
        if (L < R) continue;
        if (L > cap) { free(rd); free(sol); rd = (char *)malloc(L); sol = (uint8_t *)malloc(L); cap = L; }
        for (uint64_t j = 0; j < L; ++j) { char c = bases[offsets[r] + j]; rd[j] = (c >= 'a' && c <= 'z') ? (char)(c - 'a' + 'A') : c; }
        const uint64_t nw = L - k;
        for (uint64_t i = 0; i < nw; ++i) sol[i] = find_edge(o, rd + i) >= 0;
        for (uint64_t a = 1; a + 1 < nw && st == ORC_OK;) {
            if (sol[a] || !sol[a - 1]) { ++a; continue; }
            uint64_t b = a;                                   /* run of non-solid windows a..b, x = w_{a-1} */
            while (b + 1 < nw && !sol[b + 1]) ++b;
            if (b + 1 < nw) {                                 /* y = w_{b+1} is solid */
                const char *x = rd + a - 1, *y = rd + b + 1;
                if (kmer_in(zout, nzo, k, x + 1) && kmer_in(f->aux, f->t, k, y)) {
                    for (uint64_t i = a; i <= b && st == ORC_OK; ++i) {
                        for (uint32_t t = 0; t <= k; ++t) rc[t] = comp(rd[i + k - t]);
                        st = mercy_push(m, rd + i, R);
                        if (st == ORC_OK) st = mercy_push(m, rc, R);
                    }
                }
            }
            a = b + 1;
        }
    }
    free(rd); free(sol); free(rc); free(zout);
    orc_full_free(f);
    if (st != ORC_OK) { free(m->E); free(m); return NULL; }
    return m;
}
uint64_t orc_mercy_n(const orc_mercy *m) { return m->n; }
const char *orc_mercy_edges(const orc_mercy *m) { return m->E; }
void orc_mercy_free(orc_mercy *m) { if (m) { free(m->E); free(m); } }

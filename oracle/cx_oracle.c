/*
 * cx_oracle.c -- TEST INFRASTRUCTURE ONLY.  The plain, slow, obviously-correct CPU definition of the
 * collection BWT that the CUDA path must reproduce bit for bit.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
 * this.  It shares no code, header, table or helper with paper_1401_7457_b200/ (the product), works
 * on plain ASCII reads and a real five-symbol alphabet, and knows nothing about 2-bit packing,
 * bucket codes or radix keys.
 *
 * What it computes is the DEFINITION, PAPER.md:53-55 (Section 2), written out:
 *   1. R = {S_0..S_{n-1}}, S_i over {A,C,G,T} of length m_i >= 0, followed by its own end-marker $_i.
 *   2. every suffix (i,p), 0 <= p <= m_i, is S_i[p..m_i-1] $_i            ("each string has m+1 suffixes")
 *   3. sort them lexicographically with  $ < A < C < G < T  (Figure 1 column order
 *      PAPER.md:59-65) and  $_i < $_j iff i < j
 *   4. B_R[k] = the symbol preceding the k-th suffix in its own string; '$' for a suffix that
 *      starts at position 0 (last sentence of the definition).
 * No blocking, bucketing, key packing or reordering: materialise, comparison-sort, read off
 * (Figure 2 step 3(c)iii, is the read-off).
 *
 * Readings of silent points: per-read lengths m_i may differ (A1); m_i = 0 and
 * n = 0 are legal (A2); bytes outside ACGT are rejected (A8).
 *
 * Pins (tests/test_oracle_pins.py): Figure 1 symbol for symbol, closed forms,
 * brute force on hand-enumerable collections, LF-mapping inversion, and reduction to a generic
 * integer-alphabet suffix array.  Nothing here is "parity unpinned".
 */
#define _GNU_SOURCE
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define CX_ORACLE_OK 0
#define CX_ORACLE_BAD_BASE (-1)
#define CX_ORACLE_NOMEM (-2)
#define CX_ORACLE_ARG (-3)
#define CX_ORACLE_SMALL_BUFFER (-4)

typedef struct {
    uint64_t read; /* i */
    uint64_t pos;  /* p, 0..m_i */
} cx_suffix_t;

typedef struct {
    const uint8_t *text;     /* reads back to back, ASCII, no terminators stored */
    const uint64_t *offsets; /* n+1 base offsets */
} cx_ctx_t;

/* rank of a symbol under $ < A < C < G < T; -1 for anything else */
static int symbol_rank(uint8_t c) {
    switch (c) {
    case '$': return 0;
    case 'A': return 1;
    case 'C': return 2;
    case 'G': return 3;
    case 'T': return 4;
    default: return -1;
    }
}

/* k-th symbol of suffix s: a base while inside the read, the end-marker (rank 0) at position m_i */
static int suffix_symbol_rank(const cx_ctx_t *c, const cx_suffix_t *s, uint64_t k, int *is_end) {
    uint64_t len = c->offsets[s->read + 1] - c->offsets[s->read];
    if (s->pos + k >= len) {
        *is_end = 1;
        return 0;
    }
    *is_end = 0;
    return symbol_rank(c->text[c->offsets[s->read] + s->pos + k]);
}

/* The comparator of PAPER.md:55: first differing symbol decides; two end-markers met at the same
 * position are ordered by read index.  No comparison runs past an end-marker. */
static int compare_suffixes(const void *pa, const void *pb, void *pc) {
    const cx_suffix_t *a = (const cx_suffix_t *)pa, *b = (const cx_suffix_t *)pb;
    const cx_ctx_t *c = (const cx_ctx_t *)pc;
    for (uint64_t k = 0;; ++k) {
        int ea, eb;
        int ra = suffix_symbol_rank(c, a, k, &ea);
        int rb = suffix_symbol_rank(c, b, k, &eb);
        if (ea && eb) {
            if (a->read != b->read) return a->read < b->read ? -1 : 1;
            return 0; /* same suffix */
        }
        if (ra != rb) return ra < rb ? -1 : 1;
    }
}

static int validate(const uint8_t *text, const uint64_t *offsets, uint64_t n_reads) {
    if (n_reads && (!offsets || offsets[0] != 0)) return CX_ORACLE_ARG;
    for (uint64_t i = 0; i < n_reads; ++i)
        if (offsets[i + 1] < offsets[i]) return CX_ORACLE_ARG;
    uint64_t total = n_reads ? offsets[n_reads] : 0;
    for (uint64_t j = 0; j < total; ++j)
        if (symbol_rank(text[j]) < 1) return CX_ORACLE_BAD_BASE;
    return CX_ORACLE_OK;
}

/* symbol preceding suffix (i,p): '$' at p = 0, else S_i[p-1] */
static uint8_t preceding_symbol(const cx_ctx_t *c, const cx_suffix_t *s) {
    return s->pos == 0 ? (uint8_t)'$' : c->text[c->offsets[s->read] + s->pos - 1];
}

/*
 * Full definition.  out_bwt receives N = offsets[n] + n bytes.  If out_order is non-NULL it receives
 * the sorted suffix list as N (read, pos) pairs (2N uint64) -- used to check Figure 1's columns.
 */
int cx_oracle_bwt(const uint8_t *text, const uint64_t *offsets, uint64_t n_reads, uint8_t *out_bwt,
                  uint64_t *out_order) {
    int rc = validate(text, offsets, n_reads);
    if (rc) return rc;
    if (n_reads == 0) return CX_ORACLE_OK;
    uint64_t N = offsets[n_reads] + n_reads;
    cx_suffix_t *L = (cx_suffix_t *)malloc(N * sizeof(cx_suffix_t));
    if (!L) return CX_ORACLE_NOMEM;
    uint64_t k = 0;
    for (uint64_t i = 0; i < n_reads; ++i) {
        uint64_t m = offsets[i + 1] - offsets[i];
        for (uint64_t p = 0; p <= m; ++p) {
            L[k].read = i;
            L[k].pos = p;
            ++k;
        }
    }
    cx_ctx_t ctx = {text, offsets};
    qsort_r(L, N, sizeof(cx_suffix_t), compare_suffixes, &ctx);
    for (k = 0; k < N; ++k) {
        out_bwt[k] = preceding_symbol(&ctx, &L[k]);
        if (out_order) {
            out_order[2 * k] = L[k].read;
            out_order[2 * k + 1] = L[k].pos;
        }
    }
    free(L);
    return CX_ORACLE_OK;
}

/* -1 / 0 / +1: does suffix s sort below, inside, or above the set of suffixes that begin with the
 * base string P (|P| = plen, over ACGT)?  A suffix that ends before matching all of P is below it
 * when everything so far matched ($ is the smallest symbol). */
static int side_of_prefix(const cx_ctx_t *c, const cx_suffix_t *s, const uint8_t *P, uint64_t plen) {
    for (uint64_t k = 0; k < plen; ++k) {
        int e;
        int r = suffix_symbol_rank(c, s, k, &e);
        int rp = symbol_rank(P[k]);
        if (r != rp) return r < rp ? -1 : 1;
    }
    return 0;
}

/*
 * Range-restricted form: the same four steps applied only to the suffixes that begin with the base
 * string `prefix`.  By PAPER.md:73 ("Each partition gives a portion of the BWT, which can be simply
 * concatenated") the result is the slice B_R[slice_offset .. slice_offset + slice_len), where
 * slice_offset = number of suffixes that sort below every suffix starting with `prefix`.
 */
int cx_oracle_bwt_with_prefix(const uint8_t *text, const uint64_t *offsets, uint64_t n_reads,
                              const uint8_t *prefix, uint64_t prefix_len, uint8_t *out_slice,
                              uint64_t out_capacity, uint64_t *slice_offset, uint64_t *slice_len) {
    int rc = validate(text, offsets, n_reads);
    if (rc) return rc;
    for (uint64_t k = 0; k < prefix_len; ++k)
        if (symbol_rank(prefix[k]) < 1) return CX_ORACLE_ARG;
    cx_ctx_t ctx = {text, offsets};
    uint64_t below = 0, inside = 0;
    for (uint64_t i = 0; i < n_reads; ++i) {
        uint64_t m = offsets[i + 1] - offsets[i];
        for (uint64_t p = 0; p <= m; ++p) {
            cx_suffix_t s = {i, p};
            int side = side_of_prefix(&ctx, &s, prefix, prefix_len);
            below += side < 0;
            inside += side == 0;
        }
    }
    *slice_offset = below;
    *slice_len = inside;
    if (inside > out_capacity) return CX_ORACLE_SMALL_BUFFER;
    if (inside == 0) return CX_ORACLE_OK;
    cx_suffix_t *L = (cx_suffix_t *)malloc(inside * sizeof(cx_suffix_t));
    if (!L) return CX_ORACLE_NOMEM;
    uint64_t k = 0;
    for (uint64_t i = 0; i < n_reads; ++i) {
        uint64_t m = offsets[i + 1] - offsets[i];
        for (uint64_t p = 0; p <= m; ++p) {
            cx_suffix_t s = {i, p};
            if (side_of_prefix(&ctx, &s, prefix, prefix_len) == 0) L[k++] = s;
        }
    }
    qsort_r(L, inside, sizeof(cx_suffix_t), compare_suffixes, &ctx);
    for (k = 0; k < inside; ++k) out_slice[k] = preceding_symbol(&ctx, &L[k]);
    free(L);
    return CX_ORACLE_OK;
}

/*
 * The same steps 3-4 applied to a caller-supplied list of suffixes (read, pos) instead of all of
 * them: sort the listed suffixes with the definition's comparator and read off their preceding
 * symbols.  If the list is exactly the set of suffixes that begin with some string, the output is the
 * corresponding contiguous piece of B_R.  Used by the full-size checks of configs[3..4],
 * where the listing (a linear scan) is done outside and only the reads that own a listed suffix are
 * handed over; the read indices must keep the collection's relative order (the tie-break).
 * list: n_listed pairs (read, pos), overwritten with the sorted order.
 */
int cx_oracle_bwt_of_listed(const uint8_t *text, const uint64_t *offsets, uint64_t n_reads, uint64_t *list,
                            uint64_t n_listed, uint8_t *out) {
    int rc = validate(text, offsets, n_reads);
    if (rc) return rc;
    if (n_listed && (!list || !out)) return CX_ORACLE_ARG;
    cx_ctx_t ctx = {text, offsets};
    cx_suffix_t *L = (cx_suffix_t *)list; /* two uint64 per entry, same layout */
    for (uint64_t k = 0; k < n_listed; ++k)
        if (L[k].read >= n_reads || L[k].pos > offsets[L[k].read + 1] - offsets[L[k].read]) return CX_ORACLE_ARG;
    if (n_listed) qsort_r(L, n_listed, sizeof(cx_suffix_t), compare_suffixes, &ctx);
    for (uint64_t k = 0; k < n_listed; ++k) out[k] = preceding_symbol(&ctx, &L[k]);
    return CX_ORACLE_OK;
}

/*
 * gotoh_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded-per-pair CPU oracle for the gapped-alignment stage of
 * SOAP3-dp (arXiv 1302.5507, Methods section 3): semi-global affine-gap
 * dynamic programming of a whole read R[1..n] against any sub-region T' of a window T[1..m].
 *
 * It is the paper's "straightforward" listing written out: three full
 * (m+1) x (n+1) tables M (called H here), I and D in int32 with a true minus infinity,
 * followed by a full traceback through those tables. There is no blocking, banding, packing
 * of scores, or reordering. Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this file; the CUDA path shares no code with it.
 *
 * Symbols of the paper and the names used here (DESIGN.md "Readings" R1-R3):
 *   S_MA = match, S_MI = mismatch (<= 0), S_GO = -(gap_open + gap_extend), S_GE = -gap_extend,
 *   so that a gap of k bases costs gap_open + k * gap_extend; this is forced by the base case
 *   M(0,j) = S_GO + (j-1) S_GE.
 *   paper M = H; paper I = read base R[j] against a space (CIGAR 'I', moves along j);
 *   paper D = window base T[i] against a space (CIGAR 'D', moves along i).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): brute-force enumeration of every alignment for
 * n, m <= 6; closed forms; re-scoring of the emitted CIGAR; infix edit distance special case
 * against an independently written Levenshtein DP; worked examples in tests/golden/. The local
 * variant (oracle_align_pair_local) has its own pins in tests/test_oracle_local.py.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NEG_INF (-1000000000)
#define CODE_N 4

typedef struct {
    int32_t match;       /* S_MA > 0 (>= 0 allowed)              */
    int32_t mismatch;    /* S_MI <= 0                            */
    int32_t gap_open;    /* o >= 0                               */
    int32_t gap_extend;  /* e >= 1; gap of k costs o + k*e       */
    int64_t min_sim_q;   /* llround(min_similarity * 1e6)        */
} oracle_scoring;

typedef struct {
    int32_t score, ref_start, ref_end, read_start, read_end, n_match, n_cols;
    int32_t pass;
    int32_t cigar_len;
} oracle_result;

static inline int max2(int a, int b) { return a > b ? a : b; }

/* delta(x, y) = S_MA if x == y, S_MI otherwise; N on either side is a mismatch,
 * including N against N (BASELINE.json config 5, reading R8). */
static inline int delta(const oracle_scoring* sc, uint8_t t, uint8_t r) {
    return (t < CODE_N && r < CODE_N && t == r) ? sc->match : sc->mismatch;
}

/*
 * One pair. T[0..m) window codes, R[0..n) read codes (0..3 = ACGT, 4 = N).
 * ops_out receives BAM-encoded runs ((len << 4) | op, M=0 I=1 D=2) in alignment order and must
 * hold n + m + 1 entries. last_row, if not NULL, receives H(i, n) for i = 0..m.
 * Returns 0, or -1 when out of memory.
 */
int oracle_align_pair(const uint8_t* T, int m, const uint8_t* R, int n,
                      const oracle_scoring* sc, oracle_result* res,
                      uint32_t* ops_out, int32_t* last_row)
{
    const int o = sc->gap_open, e = sc->gap_extend;
    const size_t W = (size_t)n + 1;
    int32_t* H = (int32_t*)malloc(sizeof(int32_t) * (size_t)(m + 1) * W);
    int32_t* I = (int32_t*)malloc(sizeof(int32_t) * (size_t)(m + 1) * W);
    int32_t* D = (int32_t*)malloc(sizeof(int32_t) * (size_t)(m + 1) * W);
    uint8_t* rev = (uint8_t*)malloc((size_t)n + (size_t)m + 2);
    if (!H || !I || !D || !rev) { free(H); free(I); free(D); free(rev); return -1; }
#define AT(X, i, j) X[(size_t)(i) * W + (size_t)(j)]

    /* base cases */
    for (int i = 0; i <= m; ++i) { AT(H, i, 0) = 0; AT(I, i, 0) = NEG_INF; AT(D, i, 0) = NEG_INF; }
    for (int j = 1; j <= n; ++j) {
        AT(H, 0, j) = -(o + e * j);        /* S_GO + (j-1) S_GE */
        AT(I, 0, j) = AT(H, 0, j);         /* the I recurrence applied on row 0 */
        AT(D, 0, j) = NEG_INF;
    }
    /* recurrences; loop order of the listing at */
    for (int i = 1; i <= m; ++i) {
        for (int j = 1; j <= n; ++j) {
            int vi = max2(AT(H, i, j - 1) - (o + e), AT(I, i, j - 1) - e);
            int vd = max2(AT(H, i - 1, j) - (o + e), AT(D, i - 1, j) - e);
            int vm = AT(H, i - 1, j - 1) + delta(sc, T[i - 1], R[j - 1]);
            AT(I, i, j) = vi;
            AT(D, i, j) = vd;
            AT(H, i, j) = max2(vm, max2(vi, vd));
        }
    }
    /* result: max over 1 <= i <= m of M(i, n); lowest i on ties (reading R5) */
    int best = NEG_INF, i_end = 0;
    for (int i = 1; i <= m; ++i)
        if (AT(H, i, n) > best) { best = AT(H, i, n); i_end = i; }
    if (last_row) for (int i = 0; i <= m; ++i) last_row[i] = AT(H, i, n);

    /* traceback (paper: "backtracking could be done with only tables D and M").
     * Tie rules of DESIGN.md reading R6: in state H prefer diagonal, then deletion, then
     * insertion; inside a gap test "opened here" before "extended". */
    int i = i_end, j = n, nrev = 0, n_match = 0;
    enum { ST_H, ST_D, ST_I } st = ST_H;
    while (j > 0) {
        if (st == ST_H) {
            if (i > 0 && AT(H, i, j) == AT(H, i - 1, j - 1) + delta(sc, T[i - 1], R[j - 1])) {
                rev[nrev++] = 0;
                if (T[i - 1] < CODE_N && R[j - 1] < CODE_N && T[i - 1] == R[j - 1]) ++n_match;
                --i; --j;
            } else if (i > 0 && AT(H, i, j) == AT(D, i, j)) {
                st = ST_D;
            } else {
                st = ST_I;
            }
        } else if (st == ST_D) {
            rev[nrev++] = 2;
            if (AT(D, i, j) == AT(H, i - 1, j) - (o + e)) st = ST_H;
            --i;
        } else {
            rev[nrev++] = 1;
            if (AT(I, i, j) == AT(H, i, j - 1) - (o + e)) st = ST_H;
            --j;
        }
    }
    /* reverse and run-length encode */
    int nops = 0;
    for (int k = nrev - 1; k >= 0; ) {
        int op = rev[k], len = 0;
        while (k >= 0 && rev[k] == op) { ++len; --k; }
        ops_out[nops++] = ((uint32_t)len << 4) | (uint32_t)op;
    }
    res->score = best;
    res->ref_start = i;              /* 0-based index of the first consumed window base */
    res->ref_end = i_end - 1;
    res->read_start = 0;
    res->read_end = n - 1;
    res->n_match = n_match;
    res->n_cols = nrev;
    /* similarity filter (reading R7): identity = n_match / n_cols, integer comparison */
    res->pass = ((int64_t)n_match * 1000000LL >= sc->min_sim_q * (int64_t)nrev) ? 1 : 0;
    res->cigar_len = nops;
#undef AT
    free(H); free(I); free(D); free(rev);
    return 0;
}

/*
 * LOCAL (soft-clipping) variant, SURVEY.md 8(f2). The paper names the algorithm "Smith-Waterman" and
 * speaks of soft-clipped alignments (Figure 2 legend) although its recurrences are the semi-global ones
 * above; this function is the textbook Smith-Waterman with the paper's affine gap model (reading R18):
 *     M(i,0) = M(0,j) = 0;  I, D = -inf on the borders
 *     I, D as in PAPER.md:289-291;  M(i,j) = max(0, M(i-1,j-1) + delta, I(i,j), D(i,j))
 *     S = max over 1 <= i <= m, 1 <= j <= n of M(i,j); ties: lowest i, then lowest j.
 * Traceback from that cell with the rules of R6, stopping at the first cell with M(i,j) == 0 (tested before the
 * diagonal). read_start / read_end are the first / last aligned read base; unaligned read ends are soft clips and
 * appear in the CIGAR as BAM op 4 ('S'). n_cols counts aligned columns only. S == 0 means no alignment:
 * ref_start = 0, ref_end = -1, read_start = 0, read_end = -1, an all-'S' CIGAR, pass = 0.
 * Filter (R18): soft-clipped read bases count as columns that do not match:
 *     pass = n_cols > 0 and n_match * 1e6 >= q * (n_cols + clipped bases).
 */
int oracle_align_pair_local(const uint8_t* T, int m, const uint8_t* R, int n,
                            const oracle_scoring* sc, oracle_result* res, uint32_t* ops_out)
{
    const int o = sc->gap_open, e = sc->gap_extend;
    const size_t W = (size_t)n + 1;
    int32_t* H = (int32_t*)malloc(sizeof(int32_t) * (size_t)(m + 1) * W);
    int32_t* I = (int32_t*)malloc(sizeof(int32_t) * (size_t)(m + 1) * W);
    int32_t* D = (int32_t*)malloc(sizeof(int32_t) * (size_t)(m + 1) * W);
    uint8_t* rev = (uint8_t*)malloc((size_t)n + (size_t)m + 2);
    if (!H || !I || !D || !rev) { free(H); free(I); free(D); free(rev); return -1; }
#define AT(X, i, j) X[(size_t)(i) * W + (size_t)(j)]
    for (int i = 0; i <= m; ++i) { AT(H, i, 0) = 0; AT(I, i, 0) = NEG_INF; AT(D, i, 0) = NEG_INF; }
    for (int j = 1; j <= n; ++j) { AT(H, 0, j) = 0; AT(I, 0, j) = NEG_INF; AT(D, 0, j) = NEG_INF; }
    int best = 0, i_end = 0, j_end = 0;
    for (int i = 1; i <= m; ++i) {
        for (int j = 1; j <= n; ++j) {
            int vi = max2(AT(H, i, j - 1) - (o + e), AT(I, i, j - 1) - e);
            int vd = max2(AT(H, i - 1, j) - (o + e), AT(D, i - 1, j) - e);
            int vm = AT(H, i - 1, j - 1) + delta(sc, T[i - 1], R[j - 1]);
            AT(I, i, j) = vi;
            AT(D, i, j) = vd;
            AT(H, i, j) = max2(0, max2(vm, max2(vi, vd)));
            if (AT(H, i, j) > best) { best = AT(H, i, j); i_end = i; j_end = j; }   /* row-major scan: lowest i, then lowest j */
        }
    }
    int i = i_end, j = j_end, nrev = 0, n_match = 0;
    enum { ST_H, ST_D, ST_I } st = ST_H;
    while (best > 0) {
        if (st == ST_H) {
            if (AT(H, i, j) == 0) break;
            if (AT(H, i, j) == AT(H, i - 1, j - 1) + delta(sc, T[i - 1], R[j - 1])) {
                rev[nrev++] = 0;
                if (T[i - 1] < CODE_N && R[j - 1] < CODE_N && T[i - 1] == R[j - 1]) ++n_match;
                --i; --j;
            } else if (AT(H, i, j) == AT(D, i, j)) {
                st = ST_D;
            } else {
                st = ST_I;
            }
        } else if (st == ST_D) {
            rev[nrev++] = 2;
            if (AT(D, i, j) == AT(H, i - 1, j) - (o + e)) st = ST_H;
            --i;
        } else {
            rev[nrev++] = 1;
            if (AT(I, i, j) == AT(H, i, j - 1) - (o + e)) st = ST_H;
            --j;
        }
    }
    int nops = 0;
    const int lead = (best > 0) ? j : n, trail = (best > 0) ? n - j_end : 0;
    if (lead > 0) ops_out[nops++] = ((uint32_t)lead << 4) | 4u;
    for (int k = nrev - 1; k >= 0; ) {
        int op = rev[k], len = 0;
        while (k >= 0 && rev[k] == op) { ++len; --k; }
        ops_out[nops++] = ((uint32_t)len << 4) | (uint32_t)op;
    }
    if (trail > 0) ops_out[nops++] = ((uint32_t)trail << 4) | 4u;
    res->score = best;
    if (best > 0) { res->ref_start = i; res->ref_end = i_end - 1; res->read_start = j; res->read_end = j_end - 1; }
    else          { res->ref_start = 0; res->ref_end = -1; res->read_start = 0; res->read_end = -1; }
    res->n_match = n_match;
    res->n_cols = nrev;
    res->pass = (nrev > 0 && (int64_t)n_match * 1000000LL >= sc->min_sim_q * (int64_t)(nrev + lead + trail)) ? 1 : 0;
    res->cigar_len = nops;
#undef AT
    free(H); free(I); free(D); free(rev);
    return 0;
}

/* ---- batch interface over the same packed arrays the C-ABI library consumes ------------- */

/* base k of a 2-bit packed buffer: bits 2*(k mod 16) (LSB first) of little-endian word k/16 */
static inline uint8_t get_base(const uint32_t* packed, const uint32_t* nmask, uint64_t k) {
    if (nmask && ((nmask[k >> 5] >> (k & 31)) & 1u)) return CODE_N;
    return (uint8_t)((packed[k >> 4] >> (2 * (k & 15))) & 3u);
}

typedef struct {
    uint32_t* ops; size_t len, cap;
} opvec;

typedef struct oracle_batch {
    uint64_t n_pairs, n_ops;
    uint32_t* ops;          /* compacted, caller pair order */
} oracle_batch;

/*
 * Align pairs[0..n_pairs) with up to n_threads OpenMP threads over disjoint contiguous pair
 * ranges; the per-pair code above stays single-threaded. Per-pair outputs are written to the
 * caller's arrays (length n_pairs each); CIGAR runs are kept inside the returned handle.
 * Returns NULL on allocation failure. *threads_used receives the thread count actually used.
 */
oracle_batch* oracle_align_batch_mode(
    const uint32_t* reads_packed, const uint64_t* read_off, const uint32_t* read_len, const uint32_t* read_nmask,
    const uint32_t* wins_packed, const uint64_t* win_off, const uint32_t* win_len, const uint32_t* win_nmask,
    const uint32_t* pairs, uint64_t n_pairs, const oracle_scoring* sc, int n_threads, int local_mode,
    int32_t* score, int32_t* ref_start, int32_t* ref_end, int32_t* read_start, int32_t* read_end,
    uint8_t* pass, int32_t* n_match, int32_t* n_cols, uint64_t* cigar_off, uint32_t* cigar_len,
    int32_t* threads_used)
{
    if (n_threads < 1) n_threads = 1;
    if ((uint64_t)n_threads > n_pairs && n_pairs > 0) n_threads = (int)n_pairs;
    opvec* vecs = (opvec*)calloc((size_t)n_threads, sizeof(opvec));
    oracle_batch* b = (oracle_batch*)calloc(1, sizeof(oracle_batch));
    int failed = 0;
    if (!vecs || !b) { free(vecs); free(b); return NULL; }
    if (threads_used) *threads_used = n_threads;

#ifdef _OPENMP
#pragma omp parallel num_threads(n_threads)
#endif
    {
#ifdef _OPENMP
        int tid = omp_get_thread_num();
        int nth = omp_get_num_threads();
#else
        int tid = 0, nth = 1;
#endif
        if (tid < n_threads) {
            if (nth > n_threads) nth = n_threads;
            uint64_t lo = n_pairs * (uint64_t)tid / (uint64_t)nth;
            uint64_t hi = n_pairs * (uint64_t)(tid + 1) / (uint64_t)nth;
            opvec* v = &vecs[tid];
            uint8_t *T = NULL, *R = NULL; uint32_t* ops = NULL; size_t capT = 0, capR = 0, capO = 0;
            for (uint64_t p = lo; p < hi && !failed; ++p) {
                uint32_t ri = pairs[2 * p], wi = pairs[2 * p + 1];
                int n = (int)read_len[ri], m = (int)win_len[wi];
                if ((size_t)m > capT) { free(T); capT = (size_t)m * 2; T = (uint8_t*)malloc(capT); }
                if ((size_t)n > capR) { free(R); capR = (size_t)n * 2; R = (uint8_t*)malloc(capR); }
                if ((size_t)(n + m + 3) > capO) { free(ops); capO = (size_t)(n + m + 3) * 2; ops = (uint32_t*)malloc(capO * 4); }
                if (!T || !R || !ops) { failed = 1; break; }
                for (int k = 0; k < m; ++k) T[k] = get_base(wins_packed, win_nmask, win_off[wi] + (uint64_t)k);
                for (int k = 0; k < n; ++k) R[k] = get_base(reads_packed, read_nmask, read_off[ri] + (uint64_t)k);
                oracle_result r;
                if ((local_mode ? oracle_align_pair_local(T, m, R, n, sc, &r, ops)
                                : oracle_align_pair(T, m, R, n, sc, &r, ops, NULL)) != 0) { failed = 1; break; }
                score[p] = r.score; ref_start[p] = r.ref_start; ref_end[p] = r.ref_end;
                read_start[p] = r.read_start; read_end[p] = r.read_end;
                pass[p] = (uint8_t)r.pass; n_match[p] = r.n_match; n_cols[p] = r.n_cols;
                cigar_len[p] = (uint32_t)r.cigar_len;
                if (v->len + (size_t)r.cigar_len > v->cap) {
                    size_t nc = (v->cap ? v->cap * 2 : 1024) + (size_t)r.cigar_len;
                    uint32_t* q = (uint32_t*)realloc(v->ops, nc * 4);
                    if (!q) { failed = 1; break; }
                    v->ops = q; v->cap = nc;
                }
                memcpy(v->ops + v->len, ops, (size_t)r.cigar_len * 4);
                v->len += (size_t)r.cigar_len;
            }
            free(T); free(R); free(ops);
        }
    }
    if (!failed) {
        uint64_t tot = 0;
        for (uint64_t p = 0; p < n_pairs; ++p) { cigar_off[p] = tot; tot += cigar_len[p]; }
        b->n_pairs = n_pairs; b->n_ops = tot;
        b->ops = (uint32_t*)malloc((size_t)(tot ? tot : 1) * 4);
        if (!b->ops) failed = 1;
        else {
            size_t at = 0;   /* thread ranges are contiguous and ordered, so concatenation is caller order */
            for (int t = 0; t < n_threads; ++t) { memcpy(b->ops + at, vecs[t].ops, vecs[t].len * 4); at += vecs[t].len; }
        }
    }
    for (int t = 0; t < n_threads; ++t) free(vecs[t].ops);
    free(vecs);
    if (failed) { if (b) free(b->ops); free(b); return NULL; }
    return b;
}

/* the semi-global path of the paper (every caller before the local variant existed) */
oracle_batch* oracle_align_batch(
    const uint32_t* reads_packed, const uint64_t* read_off, const uint32_t* read_len, const uint32_t* read_nmask,
    const uint32_t* wins_packed, const uint64_t* win_off, const uint32_t* win_len, const uint32_t* win_nmask,
    const uint32_t* pairs, uint64_t n_pairs, const oracle_scoring* sc, int n_threads,
    int32_t* score, int32_t* ref_start, int32_t* ref_end, int32_t* read_start, int32_t* read_end,
    uint8_t* pass, int32_t* n_match, int32_t* n_cols, uint64_t* cigar_off, uint32_t* cigar_len,
    int32_t* threads_used)
{
    return oracle_align_batch_mode(reads_packed, read_off, read_len, read_nmask, wins_packed, win_off, win_len, win_nmask,
                                   pairs, n_pairs, sc, n_threads, 0, score, ref_start, ref_end, read_start, read_end, pass,
                                   n_match, n_cols, cigar_off, cigar_len, threads_used);
}

uint64_t oracle_batch_n_ops(const oracle_batch* b) { return b ? b->n_ops : 0; }
void oracle_batch_fetch_ops(const oracle_batch* b, uint32_t* out) { if (b && b->n_ops) memcpy(out, b->ops, (size_t)b->n_ops * 4); }
void oracle_batch_free(oracle_batch* b) { if (b) { free(b->ops); free(b); } }

/*
 * CPU ORACLE for the TCR-NET hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or helper with the CUDA path (paper_2112_06613_b200/) and
 * neither includes the other.
 *
 * What it computes is the plain definition (nothing bit-parallel, no sorting,
 * no buckets, no packing):
 *
 *   lev(a,b)  unit-cost Levenshtein distance, PAPER.md:277-293 (section II.L,
 *             Eq. 15-16; Eq. 15 is garbled in the extraction - reading Q1 in
 *             lev(i,j) = max(i,j) if min(i,j) = 0, else the minimum of
 *             lev(i-1,j)+1, lev(i,j-1)+1, lev(i-1,j-1)+[a_i != b_j]),
 *             computed "iteratively, based on a straightforward algorithm"
 *             (PAPER.md:293), i.e. the Wagner-Fischer table.
 *   edges     E = {(i,j): 0 <= i < j < N, lev(s_i,s_j) <= l_max}
 *             PAPER.md:297 (section II.M: "if and only if ... l <= l_max");
 *             one node per input row, duplicates are distinct nodes
 *             (reading Q3), no self loops (zero diagonal).
 *   CSR       the strict upper triangle of the adjacency matrix of
 *             PAPER.md:301-318 (section II.N, Eq. 17), rows ascending, columns
 *             ascending inside a row, 0-based (reading Q11).
 *   deg[u]    d(u) = sum_v A_uv, PAPER.md:224 (section II.G).
 *
 * Tier 0 evaluates the full table for every pair.  Tier 1 adds the two exact
 * prunings the paper / the definition give and nothing else:
 *   (i)  skip a pair when |m-n| > l_max  (lev >= |m-n|),
 *   (ii) the paper's own abort, PAPER.md:326 and Listing 1: stop
 *        "as soon as the smallest intermediate result exceeds" l_max, i.e.
 *        when the minimum of a finished table row is > l_max (reading Q5:
 *        the minimum is reset each row and covers j = 0..n).
 * Tier 1 is checked against tier 0 in tests/test_oracle_pins.py.
 *
 * Parity pins (none of them re-use this file's formula): see
 * tests/test_oracle_pins.py - paper's worked example ACCA/ACGG = 2
 * (PAPER.md:293), kitten/sitting = 3, closed forms, metric axioms, exhaustive
 * breadth-first search over edit scripts for all strings of length <= 5, the
 * 5-node example of PAPER.md:305-318, the l_max = 1 textbook characterisation.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC (oracle/build.py).  -O2 only - the
 * oracle is never tuned.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static inline int32_t min3(int32_t a, int32_t b, int32_t c) {
    int32_t m = a < b ? a : b;
    return m < c ? m : c;
}

/* Wagner-Fischer, full (m+1) x (n+1) table.  `D` is caller
 * scratch of at least (m+1)*(n+1) int32.  Bytes are compared for equality
 * only (reading Q8: no alphabet table). */
static int32_t lev_table(const uint8_t* a, int32_t m, const uint8_t* b, int32_t n, int32_t* D) {
    const int32_t w = n + 1;
    for (int32_t i = 0; i <= m; ++i) D[i * w] = i;          /* lev(i,0) = i */
    for (int32_t j = 0; j <= n; ++j) D[j] = j;              /* lev(0,j) = j */
    for (int32_t i = 1; i <= m; ++i)
        for (int32_t j = 1; j <= n; ++j) {
            int32_t sub = (a[i - 1] != b[j - 1]) ? 1 : 0;   /* Eq. 16 */
            D[i * w + j] = min3(D[(i - 1) * w + j] + 1,      /* deletion     */
                                D[i * w + (j - 1)] + 1,      /* insertion    */
                                D[(i - 1) * w + (j - 1)] + sub); /* substitution */
        }
    return D[m * w + n];
}

/* Same table, filled row by row, with the paper's abort:
 * returns l_max+1 as soon as a finished row has minimum > l_max. */
static int32_t lev_table_abort(const uint8_t* a, int32_t m, const uint8_t* b, int32_t n,
                               int32_t l_max, int32_t* D) {
    const int32_t w = n + 1;
    for (int32_t j = 0; j <= n; ++j) D[j] = j;
    for (int32_t i = 1; i <= m; ++i) {
        D[i * w] = i;
        int32_t min_val = D[i * w];
        for (int32_t j = 1; j <= n; ++j) {
            int32_t sub = (a[i - 1] != b[j - 1]) ? 1 : 0;
            int32_t v = min3(D[(i - 1) * w + j] + 1, D[i * w + (j - 1)] + 1,
                             D[(i - 1) * w + (j - 1)] + sub);
            D[i * w + j] = v;
            if (v < min_val) min_val = v;
        }
        if (min_val > l_max) return l_max + 1;
    }
    return D[m * w + n];
}

/* Public: one distance.  Any lengths >= 0 (reading Q7: the oracle itself has no
 * length limit).  Returns -1 if scratch cannot be allocated. */
int32_t oracle_lev(const uint8_t* a, int32_t m, const uint8_t* b, int32_t n) {
    int32_t* D = (int32_t*)malloc(sizeof(int32_t) * (size_t)(m + 1) * (size_t)(n + 1));
    if (!D) return -1;
    int32_t d = lev_table(a, m, b, n, D);
    free(D);
    return d;
}

/* Public: paper's abort variant, for the tier-1-vs-tier-0 test. */
int32_t oracle_lev_abort(const uint8_t* a, int32_t m, const uint8_t* b, int32_t n, int32_t l_max) {
    int32_t* D = (int32_t*)malloc(sizeof(int32_t) * (size_t)(m + 1) * (size_t)(n + 1));
    if (!D) return -1;
    int32_t d = lev_table_abort(a, m, b, n, l_max, D);
    free(D);
    return d;
}

typedef struct {
    int64_t* v;
    int64_t n, cap;
} vec64;

static int vec_push2(vec64* x, int64_t a, int64_t b) {
    if (x->n + 2 > x->cap) {
        int64_t cap = x->cap ? 2 * x->cap : 256;
        int64_t* p = (int64_t*)realloc(x->v, sizeof(int64_t) * (size_t)cap);
        if (!p) return -1;
        x->v = p;
        x->cap = cap;
    }
    x->v[x->n++] = a;
    x->v[x->n++] = b;
    return 0;
}

/*
 * Public: the edge set, by the double loop over i < j.
 *
 *   residues/offsets/lengths : row r is residues[offsets[r] .. offsets[r]+lengths[r])
 *   rows[0..n_rows)          : the first indices i to evaluate (ascending);
 *                              NULL means all of 0..n-1
 *   all_partners             : 0 -> partners j > i only (the edge list);
 *                              1 -> every j != i (full neighbourhood of a
 *                              sampled node, for sampled parity at large N)
 *   tier                     : 0 full table, 1 length filter + row-min abort
 *   threads                  : OpenMP threads over i (<=0: library default)
 *
 * Output: *pairs_out = malloc'd int64[2 * *n_pairs_out] of (i, j), in the loop
 * order (i ascending, then j ascending), which for all_partners = 0 is the
 * lexicographic order the CSR needs.  Free with oracle_free.  Returns 0, or -1
 * on allocation failure.  *threads_used gets the team size actually used.
 */
int oracle_edges(const uint8_t* residues, const int64_t* offsets, const int32_t* lengths, int64_t n,
                 int32_t l_max, const int64_t* rows, int64_t n_rows, int all_partners, int tier,
                 int threads, int64_t** pairs_out, int64_t* n_pairs_out, int32_t* threads_used) {
    if (!rows) n_rows = n;
    int32_t max_len = 0;
    for (int64_t r = 0; r < n; ++r)
        if (lengths[r] > max_len) max_len = lengths[r];
    vec64* per_row = (vec64*)calloc((size_t)(n_rows > 0 ? n_rows : 1), sizeof(vec64));
    if (!per_row) return -1;
    int failed = 0;
    int32_t team = 1;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#endif
#pragma omp parallel
    {
#ifdef _OPENMP
#pragma omp single
        team = omp_get_num_threads();
#endif
        int32_t* D = (int32_t*)malloc(sizeof(int32_t) * (size_t)(max_len + 1) * (size_t)(max_len + 1));
        if (!D) {
#pragma omp atomic write
            failed = 1;
        }
#pragma omp for schedule(dynamic, 1)
        for (int64_t k = 0; k < n_rows; ++k) {
            if (!D) continue;
            const int64_t i = rows ? rows[k] : k;
            const uint8_t* a = residues + offsets[i];
            const int32_t m = lengths[i];
            for (int64_t j = all_partners ? 0 : i + 1; j < n; ++j) {
                if (j == i) continue;                          /* no self loops */
                const uint8_t* b = residues + offsets[j];
                const int32_t nn = lengths[j];
                int32_t d;
                if (tier == 0) {
                    d = lev_table(a, m, b, nn, D);
                } else {
                    int32_t gap = m > nn ? m - nn : nn - m;
                    if (gap > l_max) continue;                 /* pruning (i)  */
                    d = lev_table_abort(a, m, b, nn, l_max, D); /* pruning (ii) */
                }
                if (d <= l_max) {
                    if (vec_push2(&per_row[k], i, j)) {
#pragma omp atomic write
                        failed = 1;
                    }
                }
            }
        }
        free(D);
    }
    int64_t total = 0;
    for (int64_t k = 0; k < n_rows; ++k) total += per_row[k].n;
    int64_t* out = (int64_t*)malloc(sizeof(int64_t) * (size_t)(total > 0 ? total : 1));
    if (!out) failed = 1;
    int64_t pos = 0;
    for (int64_t k = 0; k < n_rows; ++k) {
        if (!failed && per_row[k].n) memcpy(out + pos, per_row[k].v, sizeof(int64_t) * (size_t)per_row[k].n);
        pos += per_row[k].n;
        free(per_row[k].v);
    }
    free(per_row);
    if (failed) {
        free(out);
        return -1;
    }
    *pairs_out = out;
    *n_pairs_out = total / 2;
    if (threads_used) *threads_used = team;
    return 0;
}

void oracle_free(void* p) { free(p); }

/*
 * Public: the distances of a caller-supplied list of pairs, out[k] = lev(s_i, s_j) for
 * (i, j) = pairs[2k], pairs[2k+1] (the same full table as oracle_lev,
 * one pair after the other; OpenMP over the list).  Used by the parity tests to check
 * EVERY edge a large network holds (lev <= l_max) where the whole network is
 * beyond the oracle's reach.  Returns 0, or -1 on allocation failure / an index out of range.
 */
int oracle_lev_pairs(const uint8_t* residues, const int64_t* offsets, const int32_t* lengths, int64_t n,
                     const int64_t* pairs, int64_t n_pairs, int32_t* out, int threads) {
    int32_t max_len = 0;
    for (int64_t r = 0; r < n; ++r)
        if (lengths[r] > max_len) max_len = lengths[r];
    int failed = 0;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#endif
#pragma omp parallel
    {
        int32_t* D = (int32_t*)malloc(sizeof(int32_t) * (size_t)(max_len + 1) * (size_t)(max_len + 1));
        if (!D) {
#pragma omp atomic write
            failed = 1;
        }
#pragma omp for schedule(static)
        for (int64_t k = 0; k < n_pairs; ++k) {
            const int64_t i = pairs[2 * k], j = pairs[2 * k + 1];
            if (!D || i < 0 || j < 0 || i >= n || j >= n) {
#pragma omp atomic write
                failed = 1;
                continue;
            }
            out[k] = lev_table(residues + offsets[i], lengths[i], residues + offsets[j], lengths[j], D);
        }
        free(D);
    }
    return failed ? -1 : 0;
}

/*
 * Public: edge list -> CSR of the strict upper triangle + degrees
 * (PAPER.md:301-318 adjacency, PAPER.md:224 degree).  `pairs` is (i,j) with
 * i < j in lexicographic order (as oracle_edges with all_partners = 0 yields).
 * row_ptr int64[n+1], col int32[n_pairs], deg int32[n].  Returns 0, or -2 if
 * the input is not strictly increasing / has i >= j / is out of range.
 */
int oracle_csr(const int64_t* pairs, int64_t n_pairs, int64_t n, int64_t* row_ptr, int32_t* col,
               int32_t* deg) {
    for (int64_t u = 0; u <= n; ++u) row_ptr[u] = 0;
    for (int64_t u = 0; u < n; ++u) deg[u] = 0;
    for (int64_t e = 0; e < n_pairs; ++e) {
        int64_t i = pairs[2 * e], j = pairs[2 * e + 1];
        if (i < 0 || j >= n || i >= j) return -2;
        if (e > 0) {
            int64_t pi = pairs[2 * e - 2], pj = pairs[2 * e - 1];
            if (pi > i || (pi == i && pj >= j)) return -2;
        }
        row_ptr[i + 1] += 1;   /* count of row i, shifted by one */
        col[e] = (int32_t)j;
        deg[i] += 1;           /* A_ij = 1 */
        deg[j] += 1;           /* A_ji = 1 (symmetric) */
    }
    for (int64_t u = 0; u < n; ++u) row_ptr[u + 1] += row_ptr[u];
    return 0;
}

/*
 * CPU ORACLE for the network observables computed on the TCR network
 * (SURVEY.md 8(f) NEXT-1).  TEST INFRASTRUCTURE ONLY - same rules as
 * tcrnet_oracle.c: only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file; it shares
 * no code with the CUDA path.
 *
 * Every function works on the strict-upper-triangle CSR (row_ptr, col) the
 * hot path outputs and follows the definitions of
 * PAPER.md:224-232 (section II.G), 240-242 (II.H) and 254-266 (II.J) literally:
 * adjacency lists, a queue, plain loops.  No union-find, no atomics, no label
 * propagation (those are the CUDA path's techniques).
 *
 *   degree distribution  hist[d] = |{u : d(u) = d}|, so p_d = hist[d] / N and
 *                        <d> = sum_d d p_d
 *   neighbour degrees    nn_sum[u] = sum_{v in N(u)} d(v); the average neighbour
 *                        degree of the degree class d, Eq. 9:
 *                        <d_nn>(d) = sum_{d'} d' P(d'|d) with P(d'|d) the
 *                        fraction of the d * hist[d] edge ends at degree-d
 *                        nodes whose other end has degree d', i.e.
 *                        <d_nn>(d) = (sum_{u: d(u)=d} nn_sum[u]) / (d * hist[d])
 *   components           "The largest connected component (LCC) is the largest
 *                        connected subgraph": breadth-first
 *                        search from every unvisited node in ascending order, so
 *                        the label of a component is its smallest node id
 *   site percolation     "randomly choose and remove a fraction p of all ...
 *                        nodes ... while observing how ... the LCC changes"
 *                        (PAPER.md:240-242, 91); the random removal order is an
 *                        INPUT (removal_rank[u] = position of u in the order):
 *                        after N_r removals the nodes with removal_rank < N_r
 *                        are gone, with all their edges (induced subgraph,
 *                        PAPER.md:224 "subgraph")
 *   normalisations       Eq. 12: LCC(p) / ((1-p) N) = LCC / (N - N_r);
 *                        Eq. 13: Eq. 12 divided by its value at p = 0
 *
 * Readings: Q14 nested removal along one order; Q15 the
 * degree class d = 0 has <d_nn> = 0 (no neighbours; networkx convention);
 * Q16 when every node is removed Eq. 12 is 0/0 -> reported as 0.
 *
 * Pins: tests/test_observables_pins.py (networkx / scipy.sparse.csgraph as
 * independent library routines, closed forms on paths, stars, cycles, cliques,
 * the paper's 5-node example, brute-force reachability on tiny graphs).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* Symmetric adjacency lists from the upper-triangle CSR: adj_ptr[n+1], adj[2E]. */
static int build_adjacency(const int64_t* row_ptr, const int32_t* col, int64_t n, int64_t** adj_ptr_out,
                           int32_t** adj_out) {
    const int64_t e = row_ptr[n];
    int64_t* ap = (int64_t*)calloc((size_t)(n + 2), sizeof(int64_t));
    int32_t* adj = (int32_t*)malloc(sizeof(int32_t) * (size_t)(2 * e > 0 ? 2 * e : 1));
    int64_t* fill = (int64_t*)malloc(sizeof(int64_t) * (size_t)(n > 0 ? n : 1));
    if (!ap || !adj || !fill) {
        free(ap);
        free(adj);
        free(fill);
        return -1;
    }
    for (int64_t u = 0; u < n; ++u)
        for (int64_t k = row_ptr[u]; k < row_ptr[u + 1]; ++k) {
            ap[u + 1] += 1;           /* A_uv */
            ap[(int64_t)col[k] + 1] += 1; /* A_vu */
        }
    for (int64_t u = 0; u < n; ++u) ap[u + 1] += ap[u];
    for (int64_t u = 0; u < n; ++u) fill[u] = ap[u];
    for (int64_t u = 0; u < n; ++u)
        for (int64_t k = row_ptr[u]; k < row_ptr[u + 1]; ++k) {
            const int32_t v = col[k];
            adj[fill[u]++] = v;
            adj[fill[v]++] = (int32_t)u;
        }
    free(fill);
    *adj_ptr_out = ap;
    *adj_out = adj;
    return 0;
}

/* hist[0..hist_len): number of nodes of each degree.  Returns the largest
 * degree, or -2 if a degree does not fit hist_len. */
int64_t oracle_degree_histogram(const int32_t* deg, int64_t n, int64_t* hist, int64_t hist_len) {
    int64_t max_deg = 0;
    for (int64_t d = 0; d < hist_len; ++d) hist[d] = 0;
    for (int64_t u = 0; u < n; ++u) {
        if (deg[u] < 0 || deg[u] >= hist_len) return -2;
        hist[deg[u]] += 1;
        if (deg[u] > max_deg) max_deg = deg[u];
    }
    return max_deg;
}

/* nn_sum[u] = sum of the degrees of u's neighbours; class_sum[d] = sum of nn_sum
 * over the nodes of degree d; knn[d] = Eq. 9 (0 for empty classes and d = 0).
 * class_sum / knn have hist_len entries.  Returns 0, -1 (memory), -2 (range). */
int oracle_neighbor_degree(const int64_t* row_ptr, const int32_t* col, int64_t n, int64_t* nn_sum,
                           int64_t* class_sum, double* knn, int64_t hist_len) {
    int64_t* ap;
    int32_t* adj;
    if (build_adjacency(row_ptr, col, n, &ap, &adj)) return -1;
    int rc = 0;
    int64_t* cnt = (int64_t*)calloc((size_t)(hist_len > 0 ? hist_len : 1), sizeof(int64_t));
    if (!cnt) rc = -1;
    for (int64_t d = 0; d < hist_len && !rc; ++d) {
        class_sum[d] = 0;
        knn[d] = 0.0;
    }
    for (int64_t u = 0; u < n && !rc; ++u) {
        const int64_t du = ap[u + 1] - ap[u];                     /* d(u) = sum_v A_uv */
        int64_t s = 0;
        for (int64_t k = ap[u]; k < ap[u + 1]; ++k) s += ap[adj[k] + 1] - ap[adj[k]]; /* d(v) */
        nn_sum[u] = s;
        if (du >= hist_len) rc = -2;
        else {
            class_sum[du] += s;
            cnt[du] += 1;
        }
    }
    for (int64_t d = 1; d < hist_len && !rc; ++d)
        if (cnt[d] > 0) knn[d] = (double)class_sum[d] / (double)(d * cnt[d]);
    free(cnt);
    free(ap);
    free(adj);
    return rc;
}

/* Components of the subgraph induced by the nodes with alive[u] != 0 (alive ==
 * NULL: all nodes).  label[u] = smallest node id of u's component (-1 for removed
 * nodes), comp_size[u] = number of nodes of u's component (0 for removed nodes).
 * *n_components / *lcc get the number of components and the size of the largest.
 * Either output array may be NULL. */
static int components(const int64_t* ap, const int32_t* adj, int64_t n, const uint8_t* alive, int32_t* label,
                      int32_t* comp_size, int64_t* n_components, int64_t* lcc) {
    int32_t* lab = label ? label : (int32_t*)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    int32_t* queue = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    if (!lab || !queue) {
        if (!label) free(lab);
        free(queue);
        return -1;
    }
    for (int64_t u = 0; u < n; ++u) lab[u] = -1;
    if (comp_size)
        for (int64_t u = 0; u < n; ++u) comp_size[u] = 0;
    int64_t comps = 0, best = 0;
    for (int64_t s = 0; s < n; ++s) {
        if (lab[s] != -1 || (alive && !alive[s])) continue;
        int64_t head = 0, tail = 0;
        queue[tail++] = (int32_t)s;
        lab[s] = (int32_t)s;
        while (head < tail) {
            const int32_t u = queue[head++];
            for (int64_t k = ap[u]; k < ap[u + 1]; ++k) {
                const int32_t v = adj[k];
                if (lab[v] != -1 || (alive && !alive[v])) continue;
                lab[v] = (int32_t)s;
                queue[tail++] = v;
            }
        }
        if (comp_size)
            for (int64_t k = 0; k < tail; ++k) comp_size[queue[k]] = (int32_t)tail;
        comps += 1;
        if (tail > best) best = tail;
    }
    if (!label) free(lab);
    free(queue);
    *n_components = comps;
    *lcc = best;
    return 0;
}

int oracle_components(const int64_t* row_ptr, const int32_t* col, int64_t n, const uint8_t* alive, int32_t* label,
                      int32_t* comp_size, int64_t* n_components, int64_t* lcc) {
    int64_t* ap;
    int32_t* adj;
    if (build_adjacency(row_ptr, col, n, &ap, &adj)) return -1;
    const int rc = components(ap, adj, n, alive, label, comp_size, n_components, lcc);
    free(ap);
    free(adj);
    return rc;
}

/* Site percolation along one removal order.  removal_rank is a permutation of
 * 0..n-1; step k removes the n_removed[k] nodes of smallest rank (0 <= n_removed[k]
 * <= n, any order of steps).  lcc[k] = size of the LCC of what is left;
 * lcc_norm1[k] = Eq. 12, lcc_norm2[k] = Eq. 13 (either may be NULL);
 * deg_hist (may be NULL) is int64[n_steps][hist_len]: the degree histogram of
 * the remaining subgraph (removed nodes are not counted), Fig. 2(h).
 * Returns 0, -1 (memory), -2 (removal_rank is not a permutation / a degree
 * exceeds hist_len). */
int oracle_percolation(const int64_t* row_ptr, const int32_t* col, int64_t n, const int32_t* removal_rank,
                       const int64_t* n_removed, int64_t n_steps, int64_t* lcc, double* lcc_norm1,
                       double* lcc_norm2, int64_t* deg_hist, int64_t hist_len) {
    int64_t* ap;
    int32_t* adj;
    uint8_t* alive = (uint8_t*)calloc((size_t)(n > 0 ? n : 1), 1);
    if (!alive) return -1;
    for (int64_t u = 0; u < n; ++u) {                /* permutation check */
        const int32_t r = removal_rank[u];
        if (r < 0 || r >= n || alive[r]) {
            free(alive);
            return -2;
        }
        alive[r] = 1;
    }
    if (build_adjacency(row_ptr, col, n, &ap, &adj)) {
        free(alive);
        return -1;
    }
    int rc = 0;
    int64_t comps, lcc0 = 0;
    rc = components(ap, adj, n, NULL, NULL, NULL, &comps, &lcc0);   /* p = 0 for Eq. 13 */
    const double norm1_at_0 = n > 0 ? (double)lcc0 / (double)n : 0.0;
    for (int64_t k = 0; k < n_steps && !rc; ++k) {
        const int64_t nr = n_removed[k];
        if (nr < 0 || nr > n) {
            rc = -2;
            break;
        }
        for (int64_t u = 0; u < n; ++u) alive[u] = removal_rank[u] >= nr;
        int64_t best = 0;
        rc = components(ap, adj, n, alive, NULL, NULL, &comps, &best);
        if (rc) break;
        lcc[k] = best;
        const double left = (double)(n - nr);                        /* (1 - p) N */
        const double n1 = n - nr > 0 ? (double)best / left : 0.0;    /* Eq. 12 (Q16) */
        if (lcc_norm1) lcc_norm1[k] = n1;
        if (lcc_norm2) lcc_norm2[k] = norm1_at_0 > 0.0 ? n1 / norm1_at_0 : 0.0; /* Eq. 13 */
        if (deg_hist) {
            int64_t* h = deg_hist + k * hist_len;
            for (int64_t d = 0; d < hist_len; ++d) h[d] = 0;
            for (int64_t u = 0; u < n && !rc; ++u) {
                if (!alive[u]) continue;
                int64_t d = 0;
                for (int64_t q = ap[u]; q < ap[u + 1]; ++q) d += alive[adj[q]];
                if (d >= hist_len) rc = -2;
                else h[d] += 1;
            }
        }
    }
    free(ap);
    free(adj);
    free(alive);
    return rc;
}

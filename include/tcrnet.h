/*
 * tcrnet.h - C ABI of the B200-native TCR-NET hot path.
 *
 * What the library computes (PAPER.md = /root/reference/PAPER.md, arXiv 2112.06613):
 *
 *   Input   N sequences s_0..s_{N-1} over the amino-acid alphabet (PAPER.md:209-213,
 *           section II.F) and a threshold l_max in N_0.
 *   Output  the TCR network of PAPER.md:297 (section II.M): one node per input row,
 *           an undirected edge {i,j} "if and only if the Levenshtein distance l between
 *           two CDR3b sequences does not exceed a threshold value l_max (thus l <= l_max)";
 *           the Levenshtein distance is the unit-cost edit distance of PAPER.md:277-293
 *           (section II.L, Eq. 15-16).  The edge set is returned as the strict upper
 *           triangle of the adjacency matrix of PAPER.md:301-318 (section II.N, Eq. 17) in
 *           CSR form - rows i ascending, inside a row the neighbours j > i ascending,
 *           0-based - plus the node degrees d(u) = sum_v A_uv of PAPER.md:224 (section II.G).
 *           The paper names this step "the computationally most expensive task"
 *           (GPU design of the original: section II.O).
 *
 * The result is unique (no ties, no tolerance): it must equal, bit for bit, what the plain
 * double loop over a Wagner-Fischer table yields.  Readings of the paper where it is silent or
 * garbled (threshold is "<=", duplicates stay distinct nodes, no self loops, length limit 64)
 * are listed in DESIGN.md section 3.
 *
 * Conventions for every call
 *   - Return value: TCRNET_OK (0) or a negative tcrnet_status.  Nothing throws, aborts or
 *     prints.  A failed call leaves the context usable (the previous load / build, if any,
 *     may have been dropped: tcrnet_csr then returns TCRNET_ERR_STATE).
 *   - A context is bound to one CUDA device and one stream; all device work is issued on that
 *     stream.  A context is not thread-safe; different contexts are independent.
 *   - "host" / "device" in a parameter comment says which address space the pointer is in.
 *   - There is no CPU fallback: without a CUDA device tcrnet_create fails with TCRNET_ERR_CUDA.
 */
#ifndef TCRNET_H_
#define TCRNET_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define TCRNET_API __attribute__((visibility("default")))
#else
#define TCRNET_API
#endif

#define TCRNET_VERSION 100 /* 1.0.0 */
#define TCRNET_MAX_LEN 64  /* one machine word per sequence (BASELINE.json north_star) */

typedef enum tcrnet_status {
    TCRNET_OK = 0,
    TCRNET_ERR_ARG = -1,           /* NULL pointer, n < 1, unknown option, ...                 */
    TCRNET_ERR_LENGTH = -2,        /* a sequence length is 0 or > TCRNET_MAX_LEN               */
    TCRNET_ERR_RESIDUE = -3,       /* a residue byte is outside 'A'..'Z'                       */
    TCRNET_ERR_LMAX = -4,          /* l_max outside 0..TCRNET_MAX_LEN                          */
    TCRNET_ERR_STATE = -5,         /* build before load, csr/degrees before build              */
    TCRNET_ERR_NOMEM = -6,         /* the allocator returned NULL / cudaMalloc failed          */
    TCRNET_ERR_EDGE_OVERFLOW = -7, /* more edges than the configured hard limit                */
    TCRNET_ERR_CUDA = -8,          /* any other CUDA runtime error (see tcrnet_last_cuda_error)*/
    TCRNET_ERR_CAPACITY = -9       /* size beyond the fixed capacity of a no-allocation call   */
} tcrnet_status;

typedef struct tcrnet_ctx tcrnet_ctx; /* opaque */

/*
 * Device-memory allocator supplied by the caller (the Python binding backs it with
 * torch.empty(..., device="cuda"), so PyTorch's caching allocator owns every byte).
 * alloc returns a device pointer aligned to >= 256 bytes, or NULL; free releases it.
 * Both are called from the thread that calls into the library, never from a kernel.
 * Pass NULL to tcrnet_create to let the library use cudaMalloc / cudaFree.
 */
typedef struct tcrnet_allocator {
    void* (*alloc)(void* user, size_t bytes);
    void (*free)(void* user, void* ptr);
    void* user;
} tcrnet_allocator;

/* Options for tcrnet_set_option (all optional; defaults in parentheses). */
typedef enum tcrnet_option {
    TCRNET_OPT_EARLY_EXIT = 1,    /* 1: exact banded early exit on (default), 0: every column of
                                     every kept pair is computed.  Never changes the result
                                     (PAPER.md:326 describes the abort as a time saver only). */
    TCRNET_OPT_FIRST_CHECK = 2,   /* text columns processed before the first early-exit test;
                                     0 = automatic (l_max + 2, clamped to 3..8)               */
    TCRNET_OPT_EDGE_CAPACITY = 3, /* initial capacity of the edge buffer in edges; 0 = automatic
                                     (max(1 Mi, 16 N)).  The buffer grows to the exact count
                                     and the distance pass is re-run if it was too small.      */
    TCRNET_OPT_EDGE_LIMIT = 4,    /* hard limit in edges (default and maximum 2^31): beyond it
                                     tcrnet_build fails with TCRNET_ERR_EDGE_OVERFLOW          */
    TCRNET_OPT_COUNT_WORK = 5,    /* 1: the distance kernel also counts executed columns and
                                     tests (slower, for roofline accounting); default 0        */
    TCRNET_OPT_TEXT_CHUNK = 6,    /* texts per work item of the text-chunk kernel (multiple of
                                     256; default 2048)                                        */
    TCRNET_OPT_PREFIX_TRIE = 7,   /* 1 (default): bucket pairs whose early exit can act within the
                                     first 6 text columns are evaluated through the prefix trie
                                     over the sorted texts (shared prefix columns computed once,
                                     whole runs of texts skipped by one exit test); 0: every kept
                                     pair is visited by the text-chunk kernel.  Never changes the
                                     result.                                                   */
    TCRNET_OPT_TRIE_CHUNK = 8,    /* texts per work item of the prefix-trie kernel (multiple of
                                     256; default 1048576)                                    */
    TCRNET_OPT_N_QUERY = 9,       /* rectangular (query x repertoire) mode: the
                                     antigen-specific network "replaces the first N_a rows" by
                                     antigen-cognate sequences and analyses only those nodes.
                                     n_q > 0: rows 0..n_q-1 of the next tcrnet_load are the query
                                     rows and builds keep only the edges with at least one query
                                     endpoint (query-query and query-repertoire).  Through the segment
                                     join (l_max <= 6) all candidate pairs are decided and the others
                                     dropped at emission; the trie / text-chunk kernels never evaluate a
                                     pair of two non-query rows.  0 (default): all pairs.
                                     Takes effect at the next tcrnet_load.                      */
    TCRNET_OPT_DEDUP = 10,        /* 1 (default): rows with identical sequences are collapsed at
                                     load; the distance step runs over the distinct sequences and
                                     the emission multiplies every surviving pair by the rows
                                     behind it (reading Q3: one node per row, duplicates joined
                                     for every l_max >= 0).  0: every row is its own pattern /
                                     text.  Never changes the result.  Ignored (off) in the
                                     rectangular mode.  Takes effect at the next load.  A load that
                                     finds no repeated sequence makes the next seven loads of the
                                     context skip the attempt (tables of distinct clonotypes come in
                                     series; tcrnet_stats.n_distinct then reads n); setting the option
                                     again re-arms it.                                          */
    TCRNET_OPT_SEGMENT_JOIN = 11, /* exact candidate filter in front of the verification: a text cut into
                                     l_max + 1 segments shares at least one of them, unchanged and shifted by
                                     at most the edits allow, with every sequence within l_max of it; only
                                     pairs found through a hash index of the segments are verified (banded,
                                     Landau-Vishkin on per-diagonal mismatch masks).  -1 (default): used for
                                     l_max <= 6 (all-pairs mode, early exit on, TCRNET_OPT_PREFIX_TRIE on); 1: the
                                     same regardless of TCRNET_OPT_PREFIX_TRIE; 0: never (every length-compatible
                                     pair is visited through the prefix trie / text-chunk kernels).  Never changes
                                     the result.  Set it BEFORE tcrnet_load: a load made with 0 sorts the
                                     sequences lexicographically inside their length buckets (the trie needs
                                     that), any other load sorts by length only; a build that needs the trie on
                                     a load sorted by length only falls back to the text-chunk kernel.        */
    TCRNET_OPT_FAST_L1 = 12,      /* 1: builds with l_max <= 1 go through the segment join
                                     whatever TCRNET_OPT_SEGMENT_JOIN / TCRNET_OPT_PREFIX_TRIE say.  There the
                                     verification IS the textbook check - equal lengths: at most one mismatching
                                     residue (XOR of the packed codes); lengths differing by one: common prefix +
                                     common suffix cover the shorter sequence.  0 (default): no effect (the
                                     default path already takes the join).  Never changes the result.         */
    TCRNET_OPT_TIMING = 13        /* CUDA events the library records on its stream for tcrnet_stats: 0 none; 1 (default)
                                     around the distance kernels only (ms_kernel); 2 around every phase (ms_load,
                                     ms_index, ms_distance, ms_csr, ms_build too; the fields not measured read 0).
                                     An event between two short kernels costs 2-4 us and ends the programmatic
                                     launch overlap there, so level 2 makes a config-4 step about 5 % slower.     */
} tcrnet_option;

/* Work and timing of the last tcrnet_load / tcrnet_build (tcrnet_get_stats). */
typedef struct tcrnet_stats {
    int64_t n;                 /* sequences loaded                                            */
    int64_t total_len;         /* residues loaded                                             */
    int32_t min_len, max_len;  /* shortest / longest sequence                                 */
    int32_t l_max;             /* threshold of the last build                                 */
    int32_t first_check;       /* columns before the first early-exit test (0: early exit off)*/
    int64_t n_edges;           /* |E|                                                         */
    int64_t pairs_all;         /* N(N-1)/2                                                    */
    int64_t pairs_kept;        /* pairs with |len_i - len_j| <= l_max that are evaluated: of
                                  distinct sequences when the load collapsed identical rows;
                                  cells_kept / columns_kept likewise                           */
    int64_t cells_all;         /* sum over all pairs of len_i * len_j (DP cells, nominal)     */
    int64_t cells_kept;        /* same over the kept pairs                                    */
    int64_t columns_kept;      /* sum over kept pairs of the text length (nominal columns)    */
    int64_t lane_columns_exec; /* 32 x warp-level column steps executed  (COUNT_WORK only)    */
    int64_t lane_tests_exec;   /* 32 x warp-level early-exit tests executed (COUNT_WORK only) */
    int64_t lane_pairs_exec;   /* 32 x warp-level first-column steps (3-LOP3 form; COUNT_WORK) */
    int64_t lane_prefix_tests_exec; /* 32 x warp-level trie-node exit tests (COUNT_WORK only)  */
    int64_t work_items;        /* work items of the distance kernels (text-chunk kernel: one
                                  CTA of 256 patterns; prefix-trie kernel: one warp of 32)     */
    int64_t work_items_trie;   /* ... of which prefix-trie kernel                             */
    int64_t trie_nodes;        /* nodes of the prefix trie built by the last load             */
    int32_t distance_passes;   /* 1; 2 or 3 if the edge buffer / the join's verification queue had to grow */
    int32_t launches_load;     /* kernels launched by the last tcrnet_load[_device]           */
    int32_t launches_build;    /* kernels launched by the last tcrnet_build                   */
    /* times in ms from CUDA events on the context's stream; a field TCRNET_OPT_TIMING did not ask for reads 0 */
    float ms_load;             /* device time of the last load (H2D copy + pack) [TIMING 2]   */
    float ms_distance;         /* index + distance kernel(s) + emission / expansion [TIMING 2] */
    float ms_sort;             /* counting of caller-supplied keys (tcrnet_assemble), else ~0  */
    float ms_csr;              /* row_ptr / col / degrees [TIMING 2]                          */
    float ms_build;            /* whole tcrnet_build on the device [TIMING 2]                 */
    int64_t n_distinct;        /* distinct sequences among the rows (= n when TCRNET_OPT_DEDUP
                                  is off or paused, or in the rectangular mode)              */
    float ms_kernel;           /* the distance kernel launches alone (events right around them: the join's
                                  probe + verify kernels, or the trie / text-chunk kernels) [TIMING 1]  */
    float ms_index;            /* segment join: building the segment index (inside ms_distance) [TIMING 2] */
    int64_t lane_columns_live; /* unused (0)                                                     */
    int64_t join_probes;       /* segment join: directory look-ups (COUNT_WORK)                  */
    int64_t join_entries;      /* ... directory entries read (COUNT_WORK)                        */
    int64_t join_candidates;   /* ... entries that passed the composition test: their rows were fetched and
                                  the mismatch masks built (COUNT_WORK)                              */
    int64_t work_items_join;   /* work items (32 patterns x one length difference) of the join      */
    int64_t join_index_entries;/* (text, segment) entries of the index                            */
    int32_t join_mode;         /* 0: not used, 1: join + banded verification (l_max >= 2), 2: join at l_max <= 1,
                                  where the verification is the XOR / prefix-suffix check                */
    int32_t pad2_;
    int64_t join_survivors;    /* segment join: candidates that passed the filters and were verified (COUNT_WORK) */
    int64_t join_diagonals;    /* ... per-diagonal mismatch masks built, probe + verify kernels (COUNT_WORK; 0 when
                                  other distance kernels ran in the same build)                               */
    int64_t join_verified_edges; /* ... pairs of distinct sequences the verify kernel (l_max >= 2) accepted     */
    int32_t join_adapted_lengths;/* ... sequence lengths whose segment cut follows the residue statistics of the load
                                    (conserved ends) instead of the even cut                                     */
    int32_t pad3_;
} tcrnet_stats;

/*
 * Create a context on CUDA device `device` that issues all work on `cuda_stream`
 * (a cudaStream_t passed as void*; NULL = the legacy default stream).
 * `allocator` may be NULL (see above); the struct is copied.
 * Errors: TCRNET_ERR_ARG (out == NULL), TCRNET_ERR_CUDA (no such device / no driver),
 * TCRNET_ERR_NOMEM.
 */
TCRNET_API int tcrnet_create(tcrnet_ctx** out, int device, void* cuda_stream, const tcrnet_allocator* allocator);

/* Release every buffer the context owns and the context itself.  NULL is allowed. */
TCRNET_API void tcrnet_destroy(tcrnet_ctx* ctx);

/*
 * Step A1 (pack): take N sequences, validate them, copy them to the device and lay them out
 * for the distance kernels: rows collapsed to distinct sequences; stable sort into length buckets (by
 * length and row; by length, first six residues and row when TCRNET_OPT_SEGMENT_JOIN = 0, the rectangular
 * mode or TCRNET_OPT_EARLY_EXIT = 0 announce the prefix-trie kernel); permutation; per sorted position one
 * bit-plane row (5-bit residue codes, one bit of the code per word, 32 bytes up to 32 residues).  The byte / word
 * rows and the prefix trie of the trie / text-chunk kernels are built by the first build that needs them.
 * PAPER.md:326 ("each a.a. is saved as a number ... BYTE"), north_star (1).
 *
 *   residues  host, uint8[sum(lengths)]: the rows concatenated, ASCII 'A'..'Z' (any of the 26
 *             letters is a legal residue; only equality matters - DESIGN.md reading Q8)
 *   lengths   host, int32[n], each in 1..TCRNET_MAX_LEN
 *   n         1 .. 2^31-2
 *
 * Both arrays are borrowed for the duration of the call only.  Node ids of the output are the
 * caller's row indices 0..n-1; the internal sort is invisible.  Replaces any previous load and
 * drops any previous build.  Synchronises the stream.
 * Errors: ARG, LENGTH, RESIDUE, NOMEM, CUDA.
 */
TCRNET_API int tcrnet_load(tcrnet_ctx* ctx, const uint8_t* residues, const int32_t* lengths, int64_t n);

/*
 * tcrnet_load for a caller that knows the size of its residue array but has not summed the lengths (a binding that
 * was handed two arrays): residues_size >= sum(lengths) is checked block by block as the lengths are read, and no
 * byte at or beyond residues_size is ever read - TCRNET_ERR_ARG instead.  Everything else as tcrnet_load.
 */
TCRNET_API int tcrnet_load_sized(tcrnet_ctx* ctx, const uint8_t* residues, int64_t residues_size,
                                 const int32_t* lengths, int64_t n);

/*
 * Same as tcrnet_load with both arrays already in device memory (ordered on the context's
 * stream).  total_len must equal sum(lengths); it sizes the residue array.
 * The arrays are borrowed for the duration of the call only (they are re-laid out into
 * buffers the context owns).
 */
TCRNET_API int tcrnet_load_device(tcrnet_ctx* ctx, const uint8_t* residues_dev, const int32_t* lengths_dev, int64_t n,
                       int64_t total_len);

/*
 * Steps A2-A6: decide, for every unordered pair of rows, whether its Levenshtein distance
 * is <= l_max, and assemble CSR + degrees on the device.  Pairs with
 * |len_i - len_j| > l_max are never touched; for l_max <= 6 (default path) only pairs that share one of the
 * l_max + 1 segments of the longer sequence are looked at (every pair within l_max does: pigeonhole) and decided
 * exactly by a banded bit-parallel verification; otherwise every length-compatible pair goes through the
 * bit-parallel column recurrence with an exact early exit (TCRNET_OPT_SEGMENT_JOIN).  The result is the same on
 * every path.  l_max in 0..TCRNET_MAX_LEN.  May be called repeatedly on one load.
 * *n_edges_out (host, may be NULL) receives |E|.  Synchronises the stream (once: the CSR step is launched behind the
 * distance kernels on the edge count as the device holds it, into buffers reserved for TCRNET_OPT_EDGE_CAPACITY edges -
 * default max(2^20, 16 n): 28 bytes per edge of capacity; more edges than that: the buffers grow and the step repeats).
 * Errors: STATE (no load), LMAX, NOMEM, EDGE_OVERFLOW, CUDA.
 */
TCRNET_API int tcrnet_build(tcrnet_ctx* ctx, int l_max, int64_t* n_edges_out);

/*
 * Step 8(e), multi-GPU sharding: steps A2-A5 for the work items  shard + k * n_shards  only
 * (interleaved, so that every shard gets the same mix of large and small length buckets).
 * Every rank loads the same sequences and calls this with its own `shard`; the union over
 * shard = 0..n_shards-1 of the emitted keys is exactly the edge set, each edge in exactly one
 * shard.  *keys_dev (may be NULL) -> device uint64[*n_keys_out], unsorted, key = (i << 32) | j
 * with i < j the caller's row indices; owned by the context, valid until the next build /
 * assemble / restrict / load.  No CSR is produced: exchange the keys (all-gather over NCCL) and
 * call tcrnet_assemble.  Errors: ARG (shard outside 0..n_shards-1), STATE, LMAX, NOMEM,
 * EDGE_OVERFLOW, CUDA.
 */
TCRNET_API int tcrnet_build_shard(tcrnet_ctx* ctx, int l_max, int shard, int n_shards, const uint64_t** keys_dev,
                                  int64_t* n_keys_out);

/*
 * Step A6 on an edge list supplied by the caller: order the n_keys keys (i << 32) | j (device
 * uint64, any order, each edge once, i < j < n) and build CSR + degrees as tcrnet_build does
 * (PAPER.md:301-318, 224).  keys_dev is copied unless it is the pointer tcrnet_build_shard
 * returned (then it runs in place).  Errors: ARG (a key with i >= j or j >= n), STATE
 * (no load), NOMEM, EDGE_OVERFLOW, CUDA.
 */
TCRNET_API int tcrnet_assemble(tcrnet_ctx* ctx, const uint64_t* keys_dev, int64_t n_keys, int64_t* n_edges_out);

/*
 * Distance labels: *dist_dev -> device uint8[|E|], dist[e] = Levenshtein
 * distance of the two endpoints of edge e of the current CSR (aligned with
 * col).  Computed on first use after a build.  NULL when |E| = 0.  Same lifetime as tcrnet_csr.
 * Errors: ARG, STATE, NOMEM, CUDA.
 */
TCRNET_API int tcrnet_edge_distances(tcrnet_ctx* ctx, const uint8_t** dist_dev);

/*
 * Threshold sweep without re-evaluating pairs (Fig. 2(i): the largest component
 * as a function of l_max): replace the current network, built at threshold L, by the network at
 * l_max <= L, i.e. keep the edges with distance label <= l_max and rebuild row_ptr / col /
 * degrees (and the labels).  The result equals tcrnet_build(l_max) bit for bit.  May be chained
 * with decreasing l_max.  Errors: STATE (no build), LMAX (l_max < 0 or > L), NOMEM, CUDA.
 */
TCRNET_API int tcrnet_restrict(tcrnet_ctx* ctx, int l_max, int64_t* n_edges_out);

/*
 * ---- Network observables on the current CSR (what the paper does with the
 * ---- 8e5-node network, Fig. 2(f)-(h); definitions in PAPER.md section II.G-II.J) ----------------
 * All four need a built network (tcrnet_build / assemble / restrict), run on the context's stream,
 * synchronise it, and return pointers owned by the context that stay valid until the CSR changes
 * (next build / assemble / restrict / load) or the context is destroyed.  Errors: ARG, STATE,
 * NOMEM, CUDA.
 */

/*
 * Degree distribution ("the relative frequency of nodes with degree d"):
 * *hist_dev -> device int64[*max_degree_out + 1], hist[d] = number of nodes with d(u) = d, so
 * p_d = hist[d] / N and <d> = sum_d d p_d.  Either out pointer may be NULL.
 */
TCRNET_API int tcrnet_degree_histogram(tcrnet_ctx* ctx, const int64_t** hist_dev, int32_t* max_degree_out);

/*
 * Average neighbour degree (Eq. 9; Fig. 2(f)): with H = max degree + 1,
 *   *nn_sum_dev    -> device int64[n]:  sum over the neighbours v of u of d(v)  (the average neighbour
 *                     degree of node u is nn_sum[u] / d(u))
 *   *class_sum_dev -> device int64[H]:  sum of nn_sum[u] over the nodes of degree d
 *   *knn_dev       -> device double[H]: <d_nn>(d) = sum_d' d' P(d'|d) = class_sum[d] / (d * hist[d]),
 *                     one IEEE-754 division of two exactly converted integers; 0 for d = 0 and for
 *                     empty degree classes (reading Q15)
 * Any out pointer may be NULL.
 */
TCRNET_API int tcrnet_neighbor_degree(tcrnet_ctx* ctx, const int64_t** nn_sum_dev, const int64_t** class_sum_dev,
                                      const double** knn_dev);

/*
 * Connected components ("The largest connected component (LCC) is the largest
 * connected subgraph"): *label_dev -> device int32[n], label[u] = smallest node id of u's component
 * (unique); *comp_size_dev -> device int32[n], number of nodes of u's component (the cluster-size
 * distribution of PAPER.md:224 is its histogram over the nodes with label[u] == u);
 * *n_components_out, *lcc_out (host): number of components, size of the largest.  Any may be NULL.
 */
TCRNET_API int tcrnet_components(tcrnet_ctx* ctx, const int32_t** label_dev, const int32_t** comp_size_dev,
                                 int64_t* n_components_out, int64_t* lcc_out);

/*
 * Site percolation / robustness (Fig. 2(g),(h)): nodes are removed along ONE
 * removal order supplied by the caller (the method's random draw is an input: removal_rank[u] =
 * position of node u in the order, a permutation of 0..n-1; reading Q14).  Step k looks at the
 * subgraph induced by the nodes with removal_rank[u] >= n_removed[k] (p = n_removed[k] / N) and
 * reports
 *   lcc_out[k]        size of its largest connected component, LCC(p)
 *   lcc_norm1_out[k]  Eq. 12: LCC(p) / ((1 - p) N) = LCC / (N - n_removed[k]); 0 when
 *                     nothing is left (reading Q16)
 *   lcc_norm2_out[k]  Eq. 13: Eq. 12 divided by its value at p = 0
 *   deg_hist_out      int64[n_steps][max_degree + 1] (max_degree of the full network, see
 *                     tcrnet_degree_histogram): degree histogram of the remaining subgraph, Fig. 2(h)
 * removal_rank: host int32[n]; n_removed: host int64[n_steps], each in 0..n, any order; the four outputs
 * are host arrays, each may be NULL.  n_steps >= 0.  The CSR itself is not modified.
 * Errors: ARG (not a permutation, a step outside 0..n), STATE, NOMEM, CUDA.
 */
TCRNET_API int tcrnet_percolation(tcrnet_ctx* ctx, const int32_t* removal_rank, const int64_t* n_removed,
                                  int32_t n_steps, int64_t* lcc_out, double* lcc_norm1_out, double* lcc_norm2_out,
                                  int64_t* deg_hist_out);

/*
 * Borrow the CSR of the last build: *row_ptr_dev -> device int64[n+1], *col_dev -> device
 * int32[|E|] (NULL when |E| = 0).  Row i lists the neighbours j > i in ascending order;
 * row_ptr[n] = |E|.  Owned by the context, valid until the next tcrnet_build / tcrnet_load /
 * tcrnet_destroy.  Either out pointer may be NULL.  Errors: ARG, STATE.
 */
TCRNET_API int tcrnet_csr(tcrnet_ctx* ctx, const int64_t** row_ptr_dev, const int32_t** col_dev);

/*
 * Borrow the degrees of the last build: *deg_dev -> device int32[n]; deg[u] counts both
 * directions (sum(deg) = 2|E|).  Same lifetime as tcrnet_csr.
 */
TCRNET_API int tcrnet_degrees(tcrnet_ctx* ctx, const int32_t** deg_dev);

/*
 * Copy the last build to host buffers (any may be NULL to skip it): row_ptr_host int64[n+1],
 * col_host int32[|E|], deg_host int32[n].  Synchronises the stream.  Errors: STATE, CUDA.
 */
TCRNET_API int tcrnet_copy_csr(tcrnet_ctx* ctx, int64_t* row_ptr_host, int32_t* col_host, int32_t* deg_host);

/* Set a tcrnet_option.  Takes effect at the next tcrnet_build unless the option says "next tcrnet_load".
   Errors: ARG. */
TCRNET_API int tcrnet_set_option(tcrnet_ctx* ctx, int option, int64_t value);

/* Fill *out (host) with the work / timing record described above.  Errors: ARG. */
TCRNET_API int tcrnet_get_stats(tcrnet_ctx* ctx, tcrnet_stats* out);

/* Last cudaError_t seen by this context (0 if none), for diagnostics. */
TCRNET_API int tcrnet_last_cuda_error(tcrnet_ctx* ctx);

/* Static string for a tcrnet_status. */
TCRNET_API const char* tcrnet_strerror(int status);

/* TCRNET_VERSION the library was built with. */
TCRNET_API int tcrnet_version(void);

/* ---------------------------------------------------------------------------------------------
 * A call that allocates nothing - for callers that cannot call cudaMalloc: code under CUDA graph
 * capture, tight serving loops, harnesses that forbid allocation.  It needs no context.
 * ------------------------------------------------------------------------------------------- */

#define TCRNET_NOALLOC_MAX_ROWS 2097152 /* 2^21 */

/*
 * The prefix-sum step of A6 (the network as sorted adjacency lists; row u's list
 * starts where the lists of the rows before it end):
 *     row_ptr[0] = 0,  row_ptr[u + 1] = row_ptr[u] + counts[u]   for u = 0..n-1
 * computed by the kernels tcrnet_build uses for it, with their scratch (one partial sum per tile of
 * 1,024 counts) in a static device array of the library instead of allocated memory: 16 KB, held by
 * every GPU that loads the library until the process exits.  No cudaMalloc, cudaFree or allocating
 * library routine is called; inputs and outputs are the caller's.
 *
 *   counts_dev     device, int32[n], each >= 0 (edges of row u whose other endpoint is larger)
 *   n              0 .. TCRNET_NOALLOC_MAX_ROWS; beyond: TCRNET_ERR_CAPACITY, and nothing is read,
 *                  written or launched
 *   row_ptr_dev    device, int64[n + 1], written
 *   cuda_stream    a cudaStream_t (NULL: the default stream).  The two kernels are enqueued there;
 *                  the call does not synchronise: row_ptr_dev is valid once the stream gets there.
 *   cuda_error_out host, may be NULL: the cudaError_t behind a TCRNET_ERR_CUDA, else 0
 *
 * The device is the one current on the calling thread (the pointers and the stream belong to it).
 * The first call on a device looks the array's address up (cudaGetSymbolAddress; the CUDA runtime
 * may load the module then): make one call - n = 0 will do - before capturing a graph.
 * ALL calls on a device share the one array: two calls whose kernels overlap on the GPU (different
 * streams, no dependency between them) race and give wrong sums; calls on one stream, or ordered by
 * events, are fine.  Nothing in the array has to start at zero: every partial sum a call reads it
 * has written itself, whatever the previous call left.
 * Errors: ARG (n < 0, NULL pointer), CAPACITY, CUDA.
 */
TCRNET_API int tcrnet_row_ptr_noalloc(const int32_t* counts_dev, int64_t n, int64_t* row_ptr_dev, void* cuda_stream,
                                      int* cuda_error_out);

/* ---------------------------------------------------------------------------------------------
 * Diagnostics - NOT part of the method: nothing above calls it and no result depends on it.
 * bench.py uses it to print the measured pipe ceilings beside the roofline it reports.
 * ------------------------------------------------------------------------------------------- */

/*
 * Measurement aid for the roofline denominator: run a dependent-chain-
 * free microkernel of one instruction class on every SM and report thread-level operations
 * per second.  kind: 0 = LOP3 (ALU pipe), 1 = IADD3 (ALU pipe), 2 = IMAD (FMA pipe),
 * 3 = LOP3 and IMAD interleaved 1:1, 4 = POPC, 5 = the Myers column step itself on registers
 * (reports column steps per second).  *ops_per_s and *sm_clock_mhz (observed, from
 * clock64 / event time) are host pointers.  Errors: ARG, CUDA.
 */
TCRNET_API int tcrnet_probe_int32(tcrnet_ctx* ctx, int kind, double* ops_per_s, double* sm_clock_mhz);

#ifdef __cplusplus
}
#endif
#endif /* TCRNET_H_ */

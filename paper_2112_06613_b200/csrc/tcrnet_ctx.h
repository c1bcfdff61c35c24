// The context behind the opaque tcrnet_ctx of include/tcrnet.h, shared by the translation units that
// implement the C ABI (tcrnet_api.cu: load / build / CSR; observables_api.cu: network observables).
// Internal to libtcrnet_b200.so.
#pragma once

#include "tcrnet_internal.h"

using namespace tcrnet;

struct DevBuf {
    void* p = nullptr;
    size_t bytes = 0;
};

struct HostCtrl {  // pinned mirror of the small device control block
    unsigned long long hist[kNumLen];
    unsigned long long edge_count;
    unsigned long long work[8];
    unsigned long long queue[kTrieQueues];  // dynamic work queues of the trie launches (zeroed with edge_count)
    unsigned long long edge_total;    // dedup: edges between rows after the expansion of the recorded pairs
    unsigned long long cand_count;    // segment join, l_max >= 2: pairs queued for verification (zeroed with edge_count)
    unsigned long long n_huge;        // dedup: products of two heavily repeated sequences set aside by the expansion
    unsigned long long probe[3];
    uint32_t flags;
    uint32_t n_long;                  // rows queued for k_sort_long_rows
    uint32_t n_distinct;              // dedup: distinct sequences of the load
    uint32_t max_group;               // dedup: rows of the most repeated sequence
    uint32_t trie_counts[8];          // [k] = nodes of trie level k
    uint32_t trie_root[kNumLen + 1];  // [L] = first level-1 node of length bucket L (non-empty buckets)
    uint32_t pad2_;
    unsigned long long hist_u[kNumLen];  // dedup: length histogram of the distinct sequences
    unsigned long long clique_edges;     // dedup: edges among the rows of the shared sequences (known at load)
    uint32_t pos_hist[2][kPosStat][32];  // pack: residue counts at the first / last positions of a sample of the rows
};

// One packed set of sequences: all rows, or the query rows of the rectangular mode.
struct SeqSet {
    bool loaded = false;
    int64_t n = 0, total_len = 0;
    int64_t hist[kNumLen] = {};
    int min_len = 0, max_len = 0;
    LengthTable lt{};
    int pat_stride = 0;
    DevBuf perm, pat, txt, trie, planes;
    bool wide_planes = false;  // bit-plane rows of 64-bit words (the longest sequence has more than 32 residues)
    float pos_bits[2][kPosStat] = {};  // collision entropy (bits) of the residue at the first / last positions; 0: unknown
    bool lexicographic = false;  // sorted by (length, first residues): the prefix trie can be built; else by length only
    bool text_tables = false;  // txt + trie are built (on demand: only the prefix-trie / text-chunk kernels read them)
    TrieLevels trie_levels{};
    uint32_t trie_root[kNumLen + 1] = {};  // level-1 node range of bucket L: [trie_root[L], trie_root[L+1])
    int64_t trie_nodes = 0;
    // dedup.cu: the set holds the distinct sequences of n_rows rows; perm is coded (row, or kGroupFlag | uid)
    bool grouped = false;
    int64_t n_rows = 0;
    DevBuf group_start, members, uid_of;
};

struct tcrnet_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    tcrnet_allocator alloc{};
    bool has_alloc = false;
    int last_cuda = 0;
    int n_sm = 0;

    // options
    int early_exit = 1;
    int first_check_opt = 0;
    int64_t edge_capacity_opt = 0;
    int64_t edge_limit = (int64_t)1 << 31;
    int count_work = 0;
    int tchunk = 2048;
    int prefix_trie = 1;
    int trie_chunk = 1 << 20;  // in practice the whole text bucket: the top of the trie is walked once per pattern tile

    int dedup = 1;        // collapse identical sequences at load (TCRNET_OPT_DEDUP)
    // TCRNET_OPT_SEGMENT_JOIN: -1 automatic (l_max <= 6, unless TCRNET_OPT_PREFIX_TRIE = 0), 0 never, 1 whenever possible
    int segment_join = -1;
    int fast_l1 = 0;        // TCRNET_OPT_FAST_L1: l_max <= 1 builds through the join with the XOR / popcount check
    int timing = 1;         // TCRNET_OPT_TIMING: 0 no events, 1 around the distance kernels (ms_kernel), 2 every phase
    int64_t n_query = 0;  // > 0: rectangular mode (TCRNET_OPT_N_QUERY)

    // load state
    bool loaded = false;
    int64_t n = 0;
    SeqSet all, query;
    unsigned long long hist_u_host[kNumLen] = {};  // length histogram of the distinct sequences of the last collapse
    uint32_t max_group = 0;          // rows of the most repeated sequence of the current load (collapsed loads)
    int64_t clique_edges = 0;        // edges among identical rows of the current load (collapsed loads)
    int64_t row_hist[kNumLen] = {};  // length histogram of the ROWS (all.hist counts distinct sequences when grouped)
    DevBuf in_res, in_len, offsets, perm_tmp, trie_scratch;  // load scratch, kept between loads (grow-only)
    DevBuf dd_table, dd_hash, dd_rep, dd_first, dd_rank, dd_count, dd_len, dd_off, dd_offsets;  // dedup scratch

    // build state
    bool built = false;      // CSR + degrees valid
    bool have_keys = false;  // tcrnet_build_shard left unsorted keys in keys_a
    bool have_dist = false;  // edge_dist valid for the current CSR
    int built_l_max = 0;
    int64_t n_edges = 0, n_keys = 0;
    DevBuf keys_a, keys_b, radix_scratch, scan_scratch, rows, row_ptr, col, deg, row_count, long_rows;
    DevBuf expand_huge;  // dedup.cu: (pair, first output position) of the products k_expand_huge spreads over the grid
    DevBuf edge_row;  // first index of every edge of the current CSR (labels.cu; valid with edge_dist)
    DevBuf inv_perm, edge_dist, edge_dist_b, flags, flag_pos;
    // segment join (segjoin.cu): directory + entries of the current load for join_l_max, work rows
    DevBuf join_cnt, join_dir, join_entries, join_rows, join_cand, join_scan_scratch;
    int64_t join_cand_cap = 0;  // pairs the verification queue join_cand holds (uint2[cap] followed by uint8[cap])
    int dedup_pause = 0;     // loads that will not try to collapse identical rows (the last attempt found none)
    bool assembled = false;  // distance_phase has run step A6 behind its first pass (tcrnet_build) and all counts fit
    int join_adapted = 0; // lengths whose segment cut was adapted to the residue statistics (make_join_tables)
    int join_l_max = -1;  // threshold the index in join_dir / join_entries was built for (-1: none)
    uint32_t join_slots = 0;
    JoinTables join_tab{};

    // observables state (observables_api.cu); valid for the current CSR only
    bool have_hist = false, have_nn = false, have_cc = false;
    int32_t max_degree = 0;
    int64_t n_components = 0, lcc = 0;
    DevBuf obs_ctrl, deg_hist, nn_sum, class_sum, knn, cc_parent, cc_count, cc_label, cc_size;
    DevBuf perc_rank, perc_seen, perc_deg, perc_hist, perc_lcc;

    DevBuf ctrl;               // device HostCtrl
    HostCtrl* h_ctrl = nullptr;  // pinned
    cudaEvent_t ev[8] = {};
    cudaStream_t side_stream = nullptr;           // work that does not depend on the distance kernels runs beside them
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;  // (no timing: cheap)
    cudaEvent_t ev_index = nullptr;               // the index built ahead by the load (second stream) is complete
    bool index_pending = false;                   // ... and nothing on the main stream has waited for it yet
    int ahead_l_max = -1;                         // threshold of the last build that used the join (-1: none yet)
    bool side_pending = false;                    // the load left work on side_stream that nothing has waited for yet
    tcrnet_stats stats{};
};

#define TRY_CUDA(expr)                         \
    do {                                       \
        cudaError_t e__ = (expr);              \
        if (e__ != cudaSuccess) {              \
            ctx->last_cuda = (int)e__;         \
            (void)cudaGetLastError();          \
            return TCRNET_ERR_CUDA;            \
        }                                      \
    } while (0)

#define TRY(expr)                     \
    do {                              \
        int rc__ = (expr);            \
        if (rc__ != TCRNET_OK) return rc__; \
    } while (0)


// tcrnet_api.cu
void dev_free(tcrnet_ctx* ctx, DevBuf& b);
int dev_reserve(tcrnet_ctx* ctx, DevBuf& b, size_t bytes);  // at least `bytes` (contents not preserved)
void drop_observables(tcrnet_ctx* ctx);                     // the CSR changed: cached observables are stale

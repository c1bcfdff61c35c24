// Internal declarations shared by the translation units of libtcrnet_b200.so.
// Nothing here is part of the C ABI (include/tcrnet.h) and nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "tcrnet.h"

namespace tcrnet {

constexpr int kMaxLen = TCRNET_MAX_LEN;  // one machine word per sequence
constexpr int kNumLen = kMaxLen + 1;     // length buckets, indexed by length 0..64
constexpr int kNumCodes = 26;            // residue code = byte - 'A'
constexpr int kPadCode = 26;             // text padding: selects an all-zero Peq row
constexpr int kPeqRows = 27;             // 26 residue rows + the zero row
constexpr int kTQ = 256;                 // patterns per CTA of the distance kernel (8 warps)
constexpr int kTT = 64;                  // texts staged into shared memory per pipeline stage
constexpr int kSortPrefix = 6;           // residues of the lexicographic sub-order inside a length bucket
constexpr int kTrieDepth = kSortPrefix;  // levels 1..kTrieDepth of the prefix trie over each text bucket
constexpr int kTrieFan = 27;             // staging slots per trie level, indexed by residue code (0..26)
constexpr int kTrieMaxL = 4;             // the trie kernel is specialised on l_max = 0..kTrieMaxL
constexpr int kTrieTile = 32;            // patterns per work item of the trie kernel: one warp
constexpr int kTrieQueues = 8;           // dynamic work queues (one per trie launch of a distance pass)
constexpr uint32_t kGroupFlag = 0x80000000u;  // perm entry = kGroupFlag | uid: a sequence shared by several rows (dedup.cu)

// Per-length layout of the packed sequence tables (filled on the host after the histogram).
struct LengthTable {
    int32_t start[kNumLen + 1];    // first sorted position of each length bucket (+ end sentinel)
    int64_t txt_base[kNumLen + 1]; // first 32-bit word of the bucket's text rows in `txt`
    int32_t row_words[kNumLen];    // words per text row = round_up(len, 4)
};

// One (pattern bucket, text bucket) pair of the tile scheduler (step A2).
struct WorkRow {
    int64_t item_begin;  // first work item of this row (chunk kernel: one CTA, kTQ patterns; trie kernel: one warp, kTrieTile)
    int64_t txt_base;    // first word of the text bucket's rows
    int32_t p_start;     // sorted position of the first pattern (the shorter-or-equal length)
    int32_t p_count;
    int32_t t_start;     // sorted position of the first text
    int32_t t_count;
    int32_t m;           // pattern length
    int32_t n;           // text length, m <= n <= m + l_max
    int32_t row_words;   // words per text row
    int32_t n_tchunks;   // text chunks per pattern tile
    int32_t diag;        // 1: same bucket, only sorted p < t counts
    int32_t tchunk;      // texts per work item
    uint32_t root_begin; // trie kernel: the text bucket's level-1 nodes are [root_begin, root_end)
    uint32_t root_end;
};
static_assert(sizeof(WorkRow) == 64, "WorkRow is copied to the device as an array");

// One node of the prefix trie (trie.cu).  Level k holds one node per maximal run of consecutive
// texts of one length bucket that share their first k residues; the nodes of a level are stored in
// sorted-text order followed by one sentinel, so node i's ranges end where node i+1's begin.
struct TrieNode {
    uint32_t text_begin;   // sorted position of the run's first text
    uint32_t child_begin;  // first child in level k+1 (level kTrieDepth: = text_begin)
    uint32_t code;         // residue code at position k-1 of the run's texts (kPadCode past the end)
    uint32_t child_codes;  // bit c set iff a child with residue code c exists (levels < kTrieDepth)
};
static_assert(sizeof(TrieNode) == 16, "TrieNode is read with 128-bit loads");
struct TrieLevels {
    TrieNode* p[kTrieDepth + 1];  // [k] = nodes of level k, k = 1..kTrieDepth ([0] unused)
};

// Which pairs a distance launch keeps (step A5).  kPairsSelf: patterns and texts are the same
// set, every unordered pair once (same-bucket rows keep sorted p < t).  The other two are the
// passes of the rectangular (query x repertoire) mode, where at least one endpoint is a query
// row (caller's rows 0..n_query-1):
//   kPairsQueryAll  patterns = query set, texts = all rows, len_t >= len_p; a text that is itself
//                   a query is kept only if it is longer, or of equal length with the larger row id
//   kPairsAllQuery  patterns = all rows, texts = query set, len_t > len_p; patterns that are
//                   queries themselves are dropped (the pair was found by the first pass)
//   kPairsSelfQuery the rectangular mode through the segment join: patterns and texts are all rows as in kPairsSelf,
//                   and a pair is kept iff one of its rows is a query row (the join looks at so few pairs that
//                   deciding all of them and dropping the others costs less than two restricted passes)
enum PairMode : int32_t { kPairsSelf = 0, kPairsQueryAll = 1, kPairsAllQuery = 2, kPairsSelfQuery = 3 };

struct DistanceParams {
    const WorkRow* rows;
    int32_t n_rows;
    int32_t l_max;
    int32_t pat_stride;  // bytes per pattern row
    int32_t mode;        // PairMode
    int32_t n_query;     // rectangular mode: rows 0..n_query-1 of the caller are the queries
    int32_t shard;       // this launch handles the work items  shard + k * n_shards  (step 8(e))
    int32_t n_shards;
    const uint32_t* txt; // text rows: one 32-bit residue code per column, padded with kPadCode
    const uint8_t* pat;  // pattern rows: one residue code per byte, row = sorted position
    const int32_t* perm_p; // sorted position -> caller's row index, pattern set
    const int32_t* perm_t; // ... text set
    unsigned long long* edges;       // keys (min(i,j) << 32) | max(i,j)
    int32_t* row_count;              // [n]: += 1 at the smaller endpoint of every emitted edge (input of the CSR step)
    int32_t* deg;                    // [n]: += 1 at the larger endpoint
    const uint32_t* group_start;     // dedup: the rows of sequence uid are members[group_start[uid] .. group_start[uid+1])
    const int32_t* members;
    unsigned long long* edge_count;  // device counter (keeps counting beyond capacity)
    unsigned long long edge_cap;
    unsigned long long* work;        // [8], COUNT only: [0] lane-columns, [1] lane-tests (exit votes), [2] lane-first-columns,
                                     //      [3] lane-V-sets (guided expansions), [4] lane-columns of lanes still alive,
                                     //      join kernels: [5] probes, [6] directory entries read, [7] candidates checked
    const TrieNode* trie[kTrieDepth + 1];  // trie kernel: nodes of level 1..kTrieDepth ([0] unused)
    unsigned long long* queue;       // trie kernel: next unclaimed work item of this launch (zeroed before the launch)
    int64_t n_items;                 // trie kernel: work items of all shards of this launch
};

// ---- segment join (segjoin.cu): an exact candidate filter in front of the distance step ----
// If lev(r, s) <= l_max and s is cut into l_max + 1 segments, at least one segment of s occurs unchanged in r
// (l_max edits touch at most l_max segments), shifted by no more than the edits allow.  The segments of every
// text are indexed in a hash directory; every pattern probes it with the substrings that could be such a
// segment, and only the pairs found this way are verified.
constexpr int kPosStat = 32;                // residue statistics of the first / last kPosStat positions (pack.cu)
constexpr int kJoinMaxL = 6;                // the join kernels are specialised on l_max = 0..kJoinMaxL
constexpr int kJoinMaxSeg = kJoinMaxL + 1;  // segments per text: l_max + 1 <= 7
constexpr int kJoinMaxProbes = 40;          // (segment, shift) probes per length difference: 1, 3, 7, 12, 19, 27, 37
                                            // at most for l_max = 0..6 (make_join_tables checks)
struct JoinTables {
    uint8_t seg_start[kNumLen][kJoinMaxSeg + 1];  // [n][i] = first residue of segment i of a text of length n; [n][k] = n
    int8_t n_probes[kJoinMaxSeg];                 // [delta]: probes of a pattern against the texts longer by delta
    int8_t probe_seg[kJoinMaxSeg][kJoinMaxProbes];
    int8_t probe_shift[kJoinMaxSeg][kJoinMaxProbes];  // the segment starting at p in the text is looked for at p + shift
    int8_t n_seg;                                 // l_max + 1
    int8_t pad_[8 - (1 + kJoinMaxSeg) % 8];
};
// One pattern bucket of the join: a work item (one warp) is a tile of 32 patterns x ONE length difference delta
// (all its probes) against the indexed text bucket of length m + delta (t_count 0: none).
struct JoinRow {
    int64_t item_begin;   // first work item of this row; the row has ceil(p_count / 32) * (l_max + 1) of them
    int32_t p_start, p_count;
    int32_t m, pad_;
    int32_t t_start[kJoinMaxSeg];
    int32_t t_count[kJoinMaxSeg];
};
// ... as the kernel sees it (passed in the parameter block)
constexpr int kJoinMaxRows = kMaxLen;
struct JoinRowDev {
    uint32_t item_begin;
    int32_t p_start, p_count;
    uint8_t m, t_mask;  // t_mask bit delta: texts of length m + delta exist
    uint16_t pad_;
};
struct JoinIndex {
    const uint32_t* dir;  // [slots + 1]: entries of hash bucket b are [dir[b], dir[b+1])
    const uint2* entries; // (composition signature of the text, its sorted position)
    uint32_t mask;        // slots - 1 (a power of two)
};
// Bit-plane rows (pack.cu, read by segjoin.cu): sequence at sorted position s = 8 words of W (uint32_t when the set's
// longest sequence has <= 32 residues: one 32-byte sector per row; else uint64_t): words 0..4 = planes, bit j of
// plane k = bit k of the 5-bit code of residue j (zero beyond the sequence); word 5 = length; 6, 7 = 0.
constexpr int kPlaneWords = 8;

// SM count of the current device (148 on B200; cached per device): grid-stride kernels are sized in multiples of it
int device_sm_count();

// ---- launch wrappers (each returns cudaGetLastError(); *launches is incremented per kernel) ----

// scan.cu: out[i] = sum_{k<i} in[k] for i in 0..n (n+1 outputs when write_total).
// scratch must hold scan_scratch_bytes(n).
size_t scan_scratch_bytes(int64_t n);
cudaError_t exclusive_scan_i32_to_i64(const int32_t* in, int64_t* out, int64_t n, bool write_total,
                                      void* scratch, cudaStream_t s, int* launches);
cudaError_t inclusive_scan_i32_to_i64(const int32_t* in, int64_t* out, int64_t n, void* scratch, cudaStream_t s,
                                      int* launches);  // out[i] = in[0] + ... + in[i], out[n] = the total
cudaError_t exclusive_scan_u32_total(const uint32_t* in, uint32_t* out /*[n+1]*/, int64_t n, void* scratch,
                                     cudaStream_t s, int* launches);

// radix.cu: stable LSD radix sort of 64-bit keys (optional 32-bit payload) over the kRadixBits-bit digits
// (key >> shifts[p]) & (2^kRadixBits - 1), p = 0..n_passes-1 in that order.  Ping-pongs between the a and b buffers;
// *result_in_b says where the sorted sequence ends up.  scratch: radix_scratch_bytes(n).
constexpr int kRadixMaxPasses = 8;
constexpr int kRadixBits = 9;
size_t radix_scratch_bytes(int64_t n);
cudaError_t radix_sort_u64(unsigned long long* keys_a, unsigned long long* keys_b, int32_t* vals_a, int32_t* vals_b,
                           int64_t n, const int* shifts, int n_passes, void* scratch, cudaStream_t s, int* launches,
                           bool* result_in_b, bool totals_cleared = false);
// the digit totals at the head of `scratch` have to be zero when the sort starts: radix_sort_u64 clears them itself
// unless the caller did (ahead of the kernels that produce the keys, so that no memset sits between two kernels)
cudaError_t radix_clear_totals(void* scratch, cudaStream_t s);

// pack.cu
// n_dev (may be NULL): device count of rows, at most n
cudaError_t launch_length_hist(const int32_t* lengths, int64_t n, const uint32_t* n_dev,
                               unsigned long long* hist /*[kNumLen]*/, uint32_t* flags, cudaStream_t s, int* launches);
// sort key of row i: ((length - 1) << 30, invalid lengths: 0) | the first kSortPrefix residues, 5 bits each (0 = past
// the end); vals[i] = i
constexpr int kSeqKeyBits = 6 + 5 * kSortPrefix;  // length - 1 (0..63) takes 6 bits
cudaError_t launch_seq_keys(const uint8_t* residues, const int64_t* offsets, const int32_t* lengths, int64_t n,
                            unsigned long long* keys, int32_t* vals, cudaStream_t s, int* launches);
// bit-plane rows of the rows in sorted order.  group_start != NULL (collapsed load): perm holds uids on entry and is
// re-coded in place (the row of an unshared sequence, or kGroupFlag | uid)
cudaError_t launch_pack(const uint8_t* residues, const int64_t* offsets, const int32_t* lengths, int32_t* perm, int64_t n,
                        void* planes, bool wide_planes, uint32_t* flags, const uint32_t* group_start,
                        const int32_t* members, uint32_t* pos_hist /*[2][kPosStat][32], zeroed; may be NULL*/,
                        cudaStream_t s, int* launches);
// pat rows (match masks) and txt rows of the trie / text-chunk kernels from the bit-plane rows, on demand
cudaError_t launch_rows_from_planes(const void* planes, bool wide_planes, int64_t n, const LengthTable& lt, int pat_stride,
                                    uint8_t* pat, uint32_t* txt, cudaStream_t s, int* launches);

// trie.cu: prefix trie over the sorted texts (levels 1..kTrieDepth, all length buckets).
//   lcp8        : scratch, uint8[round_up(n,16) + 16]
//   tile_counts : scratch, uint32[trie_tiles(n) * 8]
//   levels.p[k] : level k, capacity trie_level_capacity(n, k) nodes (sentinel included)
//   counts      : device uint32[8]: [k] = number of nodes of level k (k = 1..kTrieDepth)
//   root        : device uint32[kNumLen + 1]: [L] = first level-1 node of length bucket L (only the
//                 entries of non-empty buckets are written)
int64_t trie_tiles(int64_t n);
int64_t trie_level_capacity(int64_t n, int level);
cudaError_t launch_trie_build(const uint32_t* txt, const LengthTable& lt, int64_t n, uint8_t* lcp8,
                              uint32_t* tile_counts, const TrieLevels& levels, uint32_t* counts, uint32_t* root,
                              cudaStream_t s, int* launches);

// dedup.cu: identical sequences collapse before the pack (see the file header for the steps)
uint32_t dedup_table_slots(int64_t n);
cudaError_t launch_dedup_find(const uint8_t* residues, const int64_t* offsets, const int32_t* lengths, int64_t n,
                              int64_t total_len, unsigned long long* table /*all ones*/, uint32_t slots,
                              unsigned long long* hash, int32_t* rep_of, uint32_t* is_first,
                              unsigned long long* hist /*[kNumLen], += lengths of the rows*/, uint32_t* flags,
                              cudaStream_t s, int* launches);
// first_rank = exclusive scan of is_first; group_count zeroed by the caller
cudaError_t launch_dedup_groups(const int32_t* rep_of, const uint32_t* first_rank, const int64_t* offsets,
                                const int32_t* lengths, int64_t n, int32_t* uid_of, uint32_t* group_count,
                                int32_t* len_u, int64_t* off_u, unsigned long long* hist_u /*[kNumLen], += lengths of
                                the distinct sequences*/,
                                unsigned long long* sort_key /*may be NULL: [uid] = key of the by-length sort*/,
                                int32_t* sort_val /*[uid] = uid*/, cudaStream_t s, int* launches);
// group_start = exclusive scan of group_count (n_u + 1 entries); group_count is consumed
// *clique_edges (zeroed) += sum over the groups of g (g - 1) / 2
cudaError_t launch_dedup_fill(const int32_t* uid_of, int64_t n, const uint32_t* group_start, uint32_t* group_count,
                              int32_t* members, unsigned long long* clique_edges, uint32_t* max_group /*zeroed: largest
                              group*/, cudaStream_t s, int* launches);
// the edges among the rows of every shared sequence (distance 0); sequences uid = shard (mod n_shards) only
cudaError_t launch_emit_cliques(const int32_t* members, const int32_t* uid_of, const uint32_t* group_start, int64_t n,
                                unsigned long long* edges, unsigned long long* edge_count, unsigned long long edge_cap,
                                int32_t* row_count, int32_t* deg, int shard, int n_shards, cudaStream_t s, int* launches);
// the recorded pairs of distinct sequences (at most entry_cap of the *n_entries_dev counted) -> edges between rows
cudaError_t launch_expand_entries(const unsigned long long* entries, const unsigned long long* n_entries_dev,
                                  unsigned long long entry_cap, const uint32_t* group_start, const int32_t* members,
                                  unsigned long long* edges, unsigned long long* edge_total, unsigned long long edge_cap,
                                  int32_t* row_count, int32_t* deg, void* huge /*16 B x huge_cap: products set aside*/,
                                  unsigned long long* n_huge /*zeroed*/, uint32_t huge_cap,
                                  bool huge_possible /*two groups may have more than 4096 pairs of rows between them*/,
                                  int n_sm, cudaStream_t s, int* launches);
// inv[row] = sorted position of the row's sequence, from the coded perm
cudaError_t launch_inverse_perm_groups(const int32_t* perm, int64_t n_u, const uint32_t* group_start,
                                       const int32_t* members, int32_t* inv, cudaStream_t s, int* launches);

// distance.cu
size_t distance_smem_bytes(bool wide, int max_row_words);
cudaError_t launch_distance(const DistanceParams& p, int64_t n_items, bool wide, int first_check,
                            bool count_work, int max_row_words, cudaStream_t s, int* launches);
// distance_trie.cu: the prefix-trie kernel
size_t distance_trie_smem_bytes(bool wide);
cudaError_t launch_distance_trie(const DistanceParams& p, int64_t n_items, bool wide, bool count_work, int n_sm,
                                 cudaStream_t s, int* launches);

// segjoin.cu
// Index of the segments of the texts at sorted positions [0, n) with length >= tab.n_seg: cnt (uint32[slots], zeroed
// by the caller) is consumed, dir gets slots + 1 offsets, entries n_entries pairs.
cudaError_t launch_join_index(const void* planes, bool wide, const LengthTable& lt, int64_t n, const JoinTables& tab,
                              uint32_t* cnt, uint32_t* dir, uint2* entries, uint32_t slots, void* scan_scratch,
                              cudaStream_t s, int* launches);
// Probe + filter (+ verification and emission for l_max <= 1); for l_max >= 2 the surviving pairs go to `cand`
// (at most cand_cap of the *cand_count counted; `rows` is HOST memory) and a second kernel verifies them
// (Landau-Vishkin on the mismatch masks of the band's diagonals) and emits.  p carries the emission fields, n_items and the shard of the launch.
cudaError_t launch_join(const DistanceParams& p, const JoinRow* rows, int n_rows, const void* planes, bool wide,
                        const JoinIndex& index, const JoinTables& tab, uint2* cand, uint8_t* cand_probe,
                        unsigned long long* cand_count, unsigned long long cand_cap, bool count_work, int n_sm,
                        cudaStream_t s, int* launches);

// labels.cu: distance labels of the final edges, threshold restriction, key validation
cudaError_t launch_inverse_perm(const int32_t* perm, int64_t n, int32_t* inv, cudaStream_t s, int* launches);
// edge_row[e] = first index of edge e of the CSR
cudaError_t launch_edge_rows(const int64_t* row_ptr, int64_t n, int32_t* edge_row, cudaStream_t s, int* launches);
// dist[e] = lev(row edge_row[e], row col[e]) from the bit-plane rows (planes.cuh)
cudaError_t launch_edge_distances(const int32_t* edge_row, const int32_t* col, int64_t n_edges, const int32_t* inv_perm,
                                  const void* planes, bool wide_planes, uint8_t* dist, cudaStream_t s, int* launches);
// flags[e] = dist[e] <= l_max (uint32 0/1)
cudaError_t launch_restrict_flags(const uint8_t* dist, int64_t n_edges, int l_max, uint32_t* flags, cudaStream_t s,
                                  int* launches);
// stable compaction of the kept edges into keys (row << 32 | col) and their labels
cudaError_t launch_restrict_compact(const int32_t* edge_row, const int32_t* col, const uint8_t* dist,
                                    int64_t n_edges, const uint32_t* flags, const uint32_t* pos /*exclusive scan*/,
                                    unsigned long long* keys_out, uint8_t* dist_out, cudaStream_t s, int* launches);
// *flag |= 1 if any key has u >= v or v >= n
cudaError_t launch_validate_keys(const unsigned long long* keys, int64_t n_keys, int64_t n, uint32_t* flag,
                                 cudaStream_t s, int* launches);

// csr.cu
// counts of caller-supplied keys: row_count[u]++, deg[v]++ (both zeroed by the caller)
cudaError_t launch_count_rows(const unsigned long long* keys, int64_t n_keys, int32_t* row_count, int32_t* deg,
                              cudaStream_t s, int* launches);
// CSR + degrees from UNSORTED keys whose counts are in row_count[u] (edges of row u; left as they are) and
// deg[v] (edges whose larger endpoint is v).  bucket: uint64[n_keys] scratch, long_rows: int32[n] scratch,
// n_long: device counter, scan_scratch: scan_scratch_bytes(n).  distinct_keys: no key occurs twice (the
// library's own edge lists; a caller's list may repeat keys).  The number of keys is n_bound (n_dev = NULL) or
// *n_dev (device; a build that assembles before the host has read the count back): if that exceeds n_bound - the
// capacity of keys, bucket and col - nothing is written and the caller repeats the step with larger buffers.
cudaError_t launch_csr_unsorted(const unsigned long long* keys, const unsigned long long* n_dev, int64_t n_bound,
                                int64_t n, int32_t* row_count, int64_t* row_ptr, unsigned long long* bucket,
                                int32_t* col, int32_t* deg, int32_t* long_rows, uint32_t* n_long, void* scan_scratch,
                                bool distinct_keys, cudaStream_t s, int* launches);
// ... its last step, for the caller to launch when *n_long (rows of more than 256 neighbours, queued in long_rows) is
// not zero: until then col holds no entries for those rows
cudaError_t launch_sort_long_rows(int64_t n, const int64_t* row_ptr, const unsigned long long* bucket, int32_t* col,
                                  const int32_t* long_rows, const uint32_t* n_long, cudaStream_t s, int* launches);
// the same from keys that are already sorted (tcrnet_restrict)
cudaError_t launch_csr(const unsigned long long* sorted_keys, int64_t n_edges, int64_t n, int64_t* row_ptr,
                       int32_t* col, int32_t* deg, cudaStream_t s, int* launches);

// observables.cu: network observables on the CSR (degree distribution, Eq. 9, components, percolation steps)
cudaError_t launch_max_degree(const int32_t* deg, int64_t n, int32_t* out /*zeroed*/, cudaStream_t s, int* launches);
// hist[d] += number of alive nodes with deg[u] = d (rank == NULL: all nodes; else alive <=> rank[u] >= threshold)
cudaError_t launch_degree_hist(const int32_t* deg, int64_t n, const int32_t* rank, int32_t threshold,
                               unsigned long long* hist /*zeroed*/, cudaStream_t s, int* launches);
// nn_sum, class_sum zeroed by the caller; knn[d] = class_sum[d] / (d * hist[d])
cudaError_t launch_neighbor_degree(const int64_t* row_ptr, const int32_t* col, const int32_t* deg, int64_t n,
                                   const unsigned long long* hist, int32_t hist_len, unsigned long long* nn_sum,
                                   unsigned long long* class_sum, double* knn, cudaStream_t s, int* launches);
// union-find over the edges with two alive ends: label[u] (may be NULL) = smallest id of u's component (-1: dead),
// count[root] = component size, *lcc = max size, *n_comp = number of components (both zeroed by the caller);
// sub_deg (may be NULL) = degrees inside the induced subgraph.
cudaError_t launch_components(const int64_t* row_ptr, const int32_t* col, int64_t n, const int32_t* rank,
                              int32_t threshold, int32_t* parent, int32_t* count, int32_t* label, int32_t* sub_deg,
                              unsigned long long* lcc, unsigned long long* n_comp, cudaStream_t s, int* launches);
cudaError_t launch_component_sizes(int64_t n, const int32_t* label, const int32_t* count, int32_t* comp_size,
                                   cudaStream_t s, int* launches);
// *flag |= 1 unless rank is a permutation of 0..n-1; seen: zeroed uint32[(n + 31) / 32]
cudaError_t launch_check_permutation(const int32_t* rank, int64_t n, uint32_t* seen, uint32_t* flag, cudaStream_t s,
                                     int* launches);

// probe.cu
cudaError_t launch_probe(int kind, int n_sm, unsigned long long* out /*[2]: ops, cycles*/, float* ms,
                         cudaStream_t s);

enum : uint32_t { kFlagBadLength = 1u, kFlagBadResidue = 2u };

}  // namespace tcrnet

// C ABI of libtcrnet_b200.so (include/tcrnet.h): context, memory, the host half of the tile
// scheduler (step A2) and the orchestration of steps A1-A6 on one CUDA stream.
#include <algorithm>
#include <cstddef>
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#include "tcrnet_ctx.h"

void dev_free(tcrnet_ctx* ctx, DevBuf& b) {
    if (b.p) {
        if (ctx->has_alloc) ctx->alloc.free(ctx->alloc.user, b.p);
        else cudaFree(b.p);
    }
    b.p = nullptr;
    b.bytes = 0;
}

// Make `b` at least `bytes` large (contents are not preserved).
int dev_reserve(tcrnet_ctx* ctx, DevBuf& b, size_t bytes) {
    if (bytes == 0) bytes = 16;
    if (b.p && b.bytes >= bytes) return TCRNET_OK;
    dev_free(ctx, b);
    void* p = nullptr;
    if (ctx->has_alloc) {
        p = ctx->alloc.alloc(ctx->alloc.user, bytes);
    } else {
        if (cudaMalloc(&p, bytes) != cudaSuccess) {
            (void)cudaGetLastError();
            p = nullptr;
        }
    }
    if (!p) return TCRNET_ERR_NOMEM;
    b.p = p;
    b.bytes = bytes;
    return TCRNET_OK;
}

void drop_observables(tcrnet_ctx* ctx) { ctx->have_hist = ctx->have_nn = ctx->have_cc = false; }

namespace {

HostCtrl* d_ctrl(tcrnet_ctx* ctx) { return static_cast<HostCtrl*>(ctx->ctrl.p); }
// Timing events cost 2-4 us each between two short kernels (and end the programmatic launch chain there), so they are
// recorded only at the level TCRNET_OPT_TIMING asks for: 1 = around the distance kernels, 2 = every phase.
cudaError_t rec(tcrnet_ctx* ctx, int i, int level) {
    return ctx->timing >= level ? cudaEventRecord(ctx->ev[i], ctx->stream) : cudaSuccess;
}
constexpr uint32_t kExpandHugeCap = 1u << 16;  // products set aside for k_expand_huge (beyond: expanded by their warp)

void drop_build(tcrnet_ctx* ctx) {
    drop_observables(ctx);
    ctx->built = false;
    ctx->have_keys = false;
    ctx->have_dist = false;
    ctx->n_edges = 0;
    ctx->n_keys = 0;
}

void drop_load(tcrnet_ctx* ctx) {
    drop_build(ctx);
    ctx->loaded = false;
    ctx->all.loaded = ctx->query.loaded = false;
    ctx->n = 0;
    ctx->clique_edges = 0;
    ctx->max_group = 0;
    ctx->join_l_max = -1;  // the segment index belongs to a load
}

// Step A1: everything after the raw arrays are in device memory.  Packs rows 0..n-1 into `set`.
// total_len < 0: not known (the query prefix of the rows); it is then taken from the histogram.
// ext_offsets != NULL: residue offset of every row (the rows need not be contiguous in d_res); else the rows are
// concatenated in order.
// pre_hist != NULL: the (validated) length histogram of the rows is already on the host.
int pack_set(tcrnet_ctx* ctx, SeqSet& set, const uint8_t* d_res, const int32_t* d_len, int64_t n, int64_t total_len,
             const int64_t* ext_offsets, const unsigned long long* pre_hist, bool code_groups, bool lexicographic,
             int* launches, bool keys_ready = false /*keys_a / perm_tmp hold the keys of the by-length sort*/) {
    set.loaded = false;
    set.grouped = false;
    set.n_rows = n;
    cudaStream_t s = ctx->stream;
    HostCtrl* dc = d_ctrl(ctx);
    // (a collapsed load arrives with the histogram and a clean control block: dedup_rows returned on any flag)
    if (!pre_hist) TRY_CUDA(cudaMemsetAsync(dc, 0, sizeof(HostCtrl), s));
    if (!pre_hist) {
        TRY_CUDA(launch_length_hist(d_len, n, nullptr, dc->hist, &dc->flags, s, launches));
        TRY_CUDA(cudaMemcpyAsync(ctx->h_ctrl, dc, sizeof(HostCtrl), cudaMemcpyDeviceToHost, s));
        TRY_CUDA(cudaStreamSynchronize(s));
        if (ctx->h_ctrl->flags & kFlagBadLength) return TCRNET_ERR_LENGTH;
        pre_hist = ctx->h_ctrl->hist;
    }
    int64_t sum = 0, cnt = 0;
    int min_len = kMaxLen, max_len = 0;
    for (int l = 0; l < kNumLen; ++l) {
        set.hist[l] = (int64_t)pre_hist[l];
        if (set.hist[l]) {
            min_len = std::min(min_len, l);
            max_len = std::max(max_len, l);
        }
        sum += set.hist[l] * l;
        cnt += set.hist[l];
    }
    if (cnt != n || (total_len >= 0 && sum != total_len)) return TCRNET_ERR_ARG;
    total_len = sum;

    // per-length layout
    LengthTable& lt = set.lt;
    int64_t pos = 0, words = 0;
    for (int l = 0; l < kNumLen; ++l) {
        lt.start[l] = (int32_t)pos;
        lt.txt_base[l] = words;
        lt.row_words[l] = (l + 3) & ~3;
        pos += set.hist[l];
        words += set.hist[l] * lt.row_words[l];
    }
    lt.start[kNumLen] = (int32_t)pos;
    lt.txt_base[kNumLen] = words;
    set.pat_stride = (max_len + 15) & ~15;
    set.wide_planes = max_len > 32;
    set.text_tables = false;
    set.trie_nodes = 0;

    // offsets, stable sort by (length, first residues, row), re-layout
    DevBuf& offsets = ctx->offsets;
    int rc = dev_reserve(ctx, offsets, sizeof(int64_t) * (size_t)(n + 1));
    if (rc == TCRNET_OK) rc = dev_reserve(ctx, ctx->scan_scratch, scan_scratch_bytes(n));
    if (rc == TCRNET_OK) rc = dev_reserve(ctx, ctx->radix_scratch, radix_scratch_bytes(n));
    if (rc == TCRNET_OK) rc = dev_reserve(ctx, ctx->keys_a, sizeof(unsigned long long) * (size_t)n);
    if (rc == TCRNET_OK) rc = dev_reserve(ctx, ctx->keys_b, sizeof(unsigned long long) * (size_t)n);
    if (rc == TCRNET_OK) rc = dev_reserve(ctx, ctx->perm_tmp, sizeof(int32_t) * (size_t)n);
    if (rc == TCRNET_OK) rc = dev_reserve(ctx, set.perm, sizeof(int32_t) * (size_t)n);
    if (rc == TCRNET_OK) rc = dev_reserve(ctx, set.planes, (size_t)n * kPlaneWords * (set.wide_planes ? 8 : 4));
    if (rc != TCRNET_OK) return rc;
    // Sort key: (length, first kSortPrefix residues, row): one composite 64-bit key per row, stable LSD
    // radix sort with the row as payload.  The sub-order inside a length bucket is free (results are mapped
    // back through perm); the lexicographic one makes the 32 patterns of a warp share their first residues
    // and puts the texts of a bucket in trie order.
    cudaError_t e = cudaSuccess;
    const int64_t* d_off = ext_offsets;
    if (!d_off) {
        e = exclusive_scan_i32_to_i64(d_len, (int64_t*)offsets.p, n, true, ctx->scan_scratch.p, s, launches);
        d_off = (const int64_t*)offsets.p;
    }
    {
        // lexicographic: all 36 key bits (4 passes of 9-bit digits); else only the digit that holds the length (the
        // segment join needs length buckets, nothing more: 1 pass)
        constexpr int kAllPasses = (kSeqKeyBits + kRadixBits - 1) / kRadixBits;
        static_assert(kRadixBits * (kAllPasses - 1) <= 5 * kSortPrefix, "the last digit holds the whole length field");
        const int n_passes = lexicographic ? kAllPasses : 1;
        int shifts[kAllPasses];
        for (int p = 0; p < n_passes; ++p) shifts[p] = lexicographic ? kRadixBits * p : kRadixBits * (kAllPasses - 1);
        // an odd number of passes ends in the b buffers: make those set.perm
        int32_t* va = (int32_t*)(n_passes & 1 ? ctx->perm_tmp.p : set.perm.p);
        int32_t* vb = (int32_t*)(n_passes & 1 ? set.perm.p : ctx->perm_tmp.p);
        if (e == cudaSuccess) e = radix_clear_totals(ctx->radix_scratch.p, s);
        if (keys_ready && (lexicographic || va != (int32_t*)ctx->perm_tmp.p)) e = cudaErrorUnknown;
        if (e == cudaSuccess && !keys_ready)
            e = launch_seq_keys(d_res, d_off, d_len, n, (unsigned long long*)ctx->keys_a.p, va, s, launches);
        bool in_b = false;
        if (e == cudaSuccess)
            e = radix_sort_u64((unsigned long long*)ctx->keys_a.p, (unsigned long long*)ctx->keys_b.p, va, vb, n, shifts,
                               n_passes, ctx->radix_scratch.p, s, launches, &in_b, true);
        if (e == cudaSuccess && n > 1 && (in_b ? vb : va) != (int32_t*)set.perm.p) e = cudaErrorUnknown;
        if (e == cudaSuccess && n == 1)  // nothing was sorted: the payload sits in va
            e = cudaMemcpyAsync(set.perm.p, va, sizeof(int32_t), cudaMemcpyDeviceToDevice, s);
        set.lexicographic = lexicographic;
    }
    if (e == cudaSuccess && code_groups && ctx->side_pending) {  // the member lists (dedup_rows, second stream) are in
        e = cudaStreamWaitEvent(s, ctx->ev_join, 0);
        ctx->side_pending = false;
    }
    if (e == cudaSuccess)
        e = launch_pack(d_res, d_off, d_len, (int32_t*)set.perm.p, n, set.planes.p, set.wide_planes, &dc->flags,
                        code_groups ? (const uint32_t*)set.group_start.p : nullptr,
                        code_groups ? (const int32_t*)set.members.p : nullptr, &dc->pos_hist[0][0][0], s, launches);
    // (the text rows and the prefix trie are built by ensure_text_tables when a build needs them)
    // (collapsed load: the pack kernel has re-coded perm from uids to rows / kGroupFlag | uid)
    if (rc == TCRNET_OK && e == cudaSuccess)
        e = cudaMemcpyAsync(&ctx->h_ctrl->flags, &dc->flags,
                            sizeof(HostCtrl) - offsetof(HostCtrl, flags), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (rc != TCRNET_OK) return rc;
    TRY_CUDA(e);
    if (ctx->h_ctrl->flags & kFlagBadResidue) return TCRNET_ERR_RESIDUE;
    // how informative the residue at each of the first / last positions is: -log2 of the probability that two sampled
    // sequences agree there (0: too few samples to tell)
    for (int d = 0; d < 2; ++d)
        for (int p = 0; p < kPosStat; ++p) {
            double tot = 0, sq = 0;
            for (int c = 0; c < 32; ++c) {
                const double v = (double)ctx->h_ctrl->pos_hist[d][p][c];
                tot += v;
                sq += v * v;
            }
            set.pos_bits[d][p] = tot >= 64 ? (float)std::max(0.01, -std::log2(sq / (tot * tot))) : 0.f;
        }
    set.n = n;
    set.total_len = total_len;
    set.min_len = min_len;
    set.max_len = max_len;
    set.loaded = true;
    return TCRNET_OK;
}

// The tables only the prefix-trie / text-chunk kernels read: pattern rows (one residue code per byte) and text rows (one
// 32-bit word per column) expanded from the bit-plane rows, and the prefix trie over the text rows (trie.cu).  Built
// when a build first schedules one of those kernels (the segment join, the default for l_max <= 6, needs neither).
int ensure_text_tables(tcrnet_ctx* ctx, SeqSet& set, int* launches) {
    if (set.text_tables) return TCRNET_OK;
    cudaStream_t s = ctx->stream;
    HostCtrl* dc = d_ctrl(ctx);
    const int64_t n = set.n;
    const LengthTable& lt = set.lt;
    TRY(dev_reserve(ctx, set.txt, sizeof(uint32_t) * (size_t)(lt.txt_base[kNumLen] + 4)));
    TRY(dev_reserve(ctx, set.pat, (size_t)n * set.pat_stride));
    TRY_CUDA(launch_rows_from_planes(set.planes.p, set.wide_planes, n, lt, set.pat_stride, (uint8_t*)set.pat.p,
                                     (uint32_t*)set.txt.p, s, launches));
    size_t node_total = 0, level_off[kTrieDepth + 1] = {};
    for (int k = 1; k <= kTrieDepth; ++k) {
        level_off[k] = node_total;
        node_total += (size_t)trie_level_capacity(n, k);
    }
    const size_t lcp_bytes = (((size_t)n + 15) & ~(size_t)15) + 256;  // keeps the tile counts aligned
    DevBuf& trie_scratch = ctx->trie_scratch;
    TRY(dev_reserve(ctx, set.trie, node_total * sizeof(TrieNode)));
    TRY(dev_reserve(ctx, trie_scratch, lcp_bytes + (size_t)trie_tiles(n) * 8 * sizeof(uint32_t)));
    for (int k = 1; k <= kTrieDepth; ++k) set.trie_levels.p[k] = (TrieNode*)set.trie.p + level_off[k];
    set.trie_levels.p[0] = nullptr;
    TRY_CUDA(cudaMemsetAsync(dc->trie_counts, 0, sizeof(dc->trie_counts) + sizeof(dc->trie_root), s));
    static_assert(offsetof(HostCtrl, trie_root) == offsetof(HostCtrl, trie_counts) + sizeof(uint32_t) * 8, "one memset");
    TRY_CUDA(launch_trie_build((const uint32_t*)set.txt.p, lt, n, (uint8_t*)trie_scratch.p,
                               (uint32_t*)((uint8_t*)trie_scratch.p + (lcp_bytes & ~(size_t)255)), set.trie_levels,
                               dc->trie_counts, dc->trie_root, s, launches));
    TRY_CUDA(cudaMemcpyAsync(ctx->h_ctrl->trie_counts, dc->trie_counts, sizeof(dc->trie_counts) + sizeof(dc->trie_root),
                             cudaMemcpyDeviceToHost, s));
    TRY_CUDA(cudaStreamSynchronize(s));
    // level-1 node range of every bucket (empty buckets get an empty range)
    set.trie_root[kNumLen] = ctx->h_ctrl->trie_counts[1];
    for (int l = kNumLen - 1; l >= 0; --l)
        set.trie_root[l] = set.hist[l] ? ctx->h_ctrl->trie_root[l] : set.trie_root[l + 1];
    set.trie_nodes = 0;
    for (int k = 1; k <= kTrieDepth; ++k) set.trie_nodes += ctx->h_ctrl->trie_counts[k];
    set.text_tables = true;
    return TCRNET_OK;
}

// Work left on the second stream (dedup_rows forks the member lists there) is waited for on the host: used on the
// paths where no kernel of the main stream will.
void join_side_stream(tcrnet_ctx* ctx) {
    if (ctx->side_pending) {
        cudaStreamSynchronize(ctx->side_stream);
        ctx->side_pending = false;
    }
}

// Step A0 (dedup.cu): the distinct sequences of the rows.  On success *n_u of them, their lengths / residue
// offsets in dd_len / dd_off, and in `set` the rows behind every distinct sequence.
int dedup_rows(tcrnet_ctx* ctx, SeqSet& set, const uint8_t* d_res, const int32_t* d_len, int64_t n, int64_t total_len,
               bool by_length_keys, int64_t* n_u, int* launches) {
    cudaStream_t s = ctx->stream;
    HostCtrl* dc = d_ctrl(ctx);
    const uint32_t slots = dedup_table_slots(n);
    TRY(dev_reserve(ctx, ctx->scan_scratch, scan_scratch_bytes(n + 1)));
    TRY(dev_reserve(ctx, ctx->dd_offsets, sizeof(int64_t) * (size_t)(n + 1)));
    TRY(dev_reserve(ctx, ctx->dd_table, sizeof(unsigned long long) * (size_t)slots));
    TRY(dev_reserve(ctx, ctx->dd_hash, sizeof(unsigned long long) * (size_t)n));
    TRY(dev_reserve(ctx, ctx->dd_rep, sizeof(int32_t) * (size_t)n));
    TRY(dev_reserve(ctx, ctx->dd_first, sizeof(uint32_t) * (size_t)n));
    TRY(dev_reserve(ctx, ctx->dd_rank, sizeof(uint32_t) * (size_t)(n + 1)));
    TRY(dev_reserve(ctx, ctx->dd_count, sizeof(uint32_t) * (size_t)(n + 1)));
    TRY(dev_reserve(ctx, ctx->dd_len, sizeof(int32_t) * (size_t)n));
    TRY(dev_reserve(ctx, ctx->dd_off, sizeof(int64_t) * (size_t)n));
    TRY(dev_reserve(ctx, set.uid_of, sizeof(int32_t) * (size_t)n));
    TRY(dev_reserve(ctx, set.group_start, sizeof(uint32_t) * (size_t)(n + 2)));
    TRY(dev_reserve(ctx, set.members, sizeof(int32_t) * (size_t)n));
    if (by_length_keys) {  // the groups kernel writes the keys of the by-length sort of pack_set (no k_seq_keys launch)
        TRY(dev_reserve(ctx, ctx->keys_a, sizeof(unsigned long long) * (size_t)n));
        TRY(dev_reserve(ctx, ctx->perm_tmp, sizeof(int32_t) * (size_t)n));
    }
    const int64_t* off = (const int64_t*)ctx->dd_offsets.p;
    uint32_t* rank = (uint32_t*)ctx->dd_rank.p;
    uint32_t* count = (uint32_t*)ctx->dd_count.p;
    // every reset first and every read-back last: nothing but kernels in between, so that each of them is scheduled
    // while its predecessor drains (launch.cuh)
    TRY_CUDA(cudaMemsetAsync(dc, 0, sizeof(HostCtrl), s));
    TRY_CUDA(cudaMemsetAsync(ctx->dd_table.p, 0xff, sizeof(unsigned long long) * (size_t)slots, s));
    TRY_CUDA(cudaMemsetAsync(count, 0, sizeof(uint32_t) * (size_t)(n + 1), s));
    TRY_CUDA(exclusive_scan_i32_to_i64(d_len, (int64_t*)ctx->dd_offsets.p, n, true, ctx->scan_scratch.p, s, launches));
    // (the insert kernel also takes the length histogram of the ROWS - nominal work - and validates the lengths)
    TRY_CUDA(launch_dedup_find(d_res, off, d_len, n, total_len, (unsigned long long*)ctx->dd_table.p, slots,
                               (unsigned long long*)ctx->dd_hash.p, (int32_t*)ctx->dd_rep.p, (uint32_t*)ctx->dd_first.p,
                               dc->hist, &dc->flags, s, launches));
    TRY_CUDA(exclusive_scan_u32_total((const uint32_t*)ctx->dd_first.p, rank, n, ctx->scan_scratch.p, s, launches));
    TRY_CUDA(launch_dedup_groups((const int32_t*)ctx->dd_rep.p, rank, off, d_len, n, (int32_t*)set.uid_of.p, count,
                                 (int32_t*)ctx->dd_len.p, (int64_t*)ctx->dd_off.p, dc->hist_u,
                                 by_length_keys ? (unsigned long long*)ctx->keys_a.p : nullptr,
                                 by_length_keys ? (int32_t*)ctx->perm_tmp.p : nullptr, s, launches));
    // (... and the groups kernel the length histogram of the distinct sequences: the pack needs no round trip of its own)
    TRY_CUDA(cudaMemcpyAsync(ctx->h_ctrl, dc, sizeof(HostCtrl), cudaMemcpyDeviceToHost, s));  // hist, hist_u, flags
    TRY_CUDA(cudaMemcpyAsync(&ctx->h_ctrl->n_distinct, rank + n, sizeof(uint32_t), cudaMemcpyDeviceToHost, s));
    // The member lists are not needed before the pack: they are filled on the second stream while the host reads the
    // counts back and the sort of the distinct sequences runs (pack_set waits for ev_join before its pack kernel).
    // group_start over n + 1 counts (the tail is zero): entry n_u is the total = n
    TRY_CUDA(cudaEventRecord(ctx->ev_fork, s));
    TRY_CUDA(cudaStreamWaitEvent(ctx->side_stream, ctx->ev_fork, 0));
    TRY_CUDA(exclusive_scan_u32_total(count, (uint32_t*)set.group_start.p, n + 1, ctx->scan_scratch.p, ctx->side_stream,
                                      launches));
    TRY_CUDA(launch_dedup_fill((const int32_t*)set.uid_of.p, n, (const uint32_t*)set.group_start.p, count,
                               (int32_t*)set.members.p, &dc->clique_edges, &dc->max_group, ctx->side_stream, launches));
    TRY_CUDA(cudaEventRecord(ctx->ev_join, ctx->side_stream));
    ctx->side_pending = true;
    TRY_CUDA(cudaStreamSynchronize(s));
    if (ctx->h_ctrl->flags & kFlagBadLength) return TCRNET_ERR_LENGTH;
    int64_t sum_len = 0;
    for (int l = 0; l < kNumLen; ++l) {
        ctx->row_hist[l] = (int64_t)ctx->h_ctrl->hist[l];
        ctx->hist_u_host[l] = ctx->h_ctrl->hist_u[l];  // (the pack clears the control block)
        sum_len += ctx->row_hist[l] * l;
    }
    // the header's contract: total_len = sum of the lengths (a shorter buffer would be read past its end by the
    // pack; the insert / lookup kernels above never touch a row that does not fit)
    if (sum_len != total_len) return TCRNET_ERR_ARG;
    *n_u = (int64_t)ctx->h_ctrl->n_distinct;
    if (*n_u < 1 || *n_u > n) return TCRNET_ERR_CUDA;
    return TCRNET_OK;
}

int build_join_index_ahead(tcrnet_ctx* ctx, int* launches);

int load_from_device(tcrnet_ctx* ctx, const uint8_t* d_res, const int32_t* d_len, int64_t n, int64_t total_len,
                     int* launches) {
    const bool rect = ctx->n_query > 0 && ctx->n_query < n;
    // Sub-order inside a length bucket: lexicographic by the first residues when the prefix-trie kernel will serve
    // the builds of this load (it walks a trie over the sorted texts); the segment join only needs the buckets.
    const bool lex = rect || !ctx->early_exit || ctx->segment_join == 0;
    int64_t n_u = n;
    // A load that found no repeated sequence makes the next kDedupPause loads of the context skip the attempt (tables
    // of distinct clonotypes come in series; the attempt costs 0.1 ms at N = 5e5 and finds nothing there).
    constexpr int kDedupPause = 7;
    const bool attempt = ctx->dedup && !rect && n >= 2 && ctx->dedup_pause == 0;
    if (ctx->dedup_pause > 0) --ctx->dedup_pause;
    bool rows_known = false;  // the collapse found nothing, but left the offsets, the histogram and the sort keys of the rows
    if (attempt) {
        const int rc_dedup = dedup_rows(ctx, ctx->all, d_res, d_len, n, total_len, /*by_length_keys=*/!lex, &n_u, launches);
        if (rc_dedup != TCRNET_OK || n_u >= n) join_side_stream(ctx);  // (nothing will wait for the member lists)
        TRY(rc_dedup);
        if (n_u < n) {
            const int rc_pack = pack_set(ctx, ctx->all, d_res, (const int32_t*)ctx->dd_len.p, n_u, -1,
                                         (const int64_t*)ctx->dd_off.p, ctx->hist_u_host, true, lex, launches,
                                         /*keys_ready=*/!lex);
            join_side_stream(ctx);
            TRY(rc_pack);
            ctx->clique_edges = (int64_t)ctx->h_ctrl->clique_edges;  // (read back with the pack's flags)
            ctx->max_group = ctx->h_ctrl->max_group;
            ctx->all.grouped = true;
            ctx->all.n_rows = n;
        } else {
            ctx->dedup_pause = kDedupPause;
            rows_known = true;
        }
    }
    if (!ctx->all.loaded || !ctx->all.grouped) {
        n_u = n;
        if (rows_known) {  // (uid = row: what dedup_rows computed per distinct sequence is per row)
            for (int l = 0; l < kNumLen; ++l) ctx->hist_u_host[l] = ctx->h_ctrl->hist[l];
            TRY(pack_set(ctx, ctx->all, d_res, d_len, n, total_len, (const int64_t*)ctx->dd_offsets.p, ctx->hist_u_host,
                         false, lex, launches, /*keys_ready=*/!lex));
        } else {
            TRY(pack_set(ctx, ctx->all, d_res, d_len, n, total_len, nullptr, nullptr, false, lex, launches));
        }
    }
    if (rect) TRY(pack_set(ctx, ctx->query, d_res, d_len, ctx->n_query, -1, nullptr, nullptr, false, lex, launches));
    if (!ctx->all.grouped)
        for (int l = 0; l < kNumLen; ++l) ctx->row_hist[l] = ctx->all.hist[l];
    ctx->stats.n_distinct = n_u;
    ctx->n = n;
    ctx->stats.n = n;
    ctx->stats.total_len = total_len;
    ctx->stats.min_len = ctx->all.min_len;
    ctx->stats.max_len = ctx->all.max_len;
    ctx->stats.trie_nodes = 0;  // (built on demand: ensure_text_tables)
    ctx->loaded = true;
    TRY(build_join_index_ahead(ctx, launches));
    return TCRNET_OK;
}


// One pass of the distance step = (pattern set, text set, which pairs to keep); each pass has up to
// four launches: {chunk kernel, trie kernel} x {32-bit, 64-bit words}.
struct Schedule {
    struct Part {
        std::vector<WorkRow> rows;
        int64_t items = 0;
        int max_rw = 4;
    };
    struct Pass {
        const SeqSet* pset = nullptr;
        const SeqSet* tset = nullptr;
        int mode = kPairsSelf;
        Part part[2][2];  // [trie][wide]
        std::vector<JoinRow> join_rows[2];  // [wide]: pattern buckets served by the segment join (segjoin.cu)
        int64_t join_items[2] = {0, 0};
    };
    std::vector<Pass> passes;
    size_t n_rows = 0;
    size_t n_join_rows = 0;
    bool use_join = false, fast_l1 = false;
};

// Segment join: where a text of length n is cut (k = l_max + 1 segments) and which (segment, shift) probes a
// pattern shorter by delta has to make (segjoin.cu has the derivation: max(|d|, i) + |d + delta| <= l_max).
// n = q k + r: every segment gets q residues and r of them one more - the two outer ones first, then inwards,
// because CDR3 sequences are least diverse at their ends (conserved first / last residues), so the outer segments
// need the extra residue most.  Any cut is exact; this one only keeps the candidate lists short.
// `set`: where its residue statistics (pack.cu) say that another cut makes the LEAST informative segment of a length
// clearly more informative (real CDR3 start CASS.. and end ..EQYF: with l_max = 1 the halves of a 15-residue text then
// hold 4 + 3 free residues, cutting one residue later gives 3.5 + 3.5), that cut is taken; *adapted counts such lengths.
bool make_join_tables(int l_max, const SeqSet* set, JoinTables& tab, int* adapted) {
    std::memset(&tab, 0, sizeof(tab));
    const int k = l_max + 1;
    tab.n_seg = (int8_t)k;
    if (adapted) *adapted = 0;
    bool have_stats = false;
    if (set)
        for (int p = 0; p < kPosStat; ++p) have_stats = have_stats || set->pos_bits[0][p] > 0.f || set->pos_bits[1][p] > 0.f;
    for (int n = 0; n < kNumLen; ++n) {
        const int q = n / k, r = n % k;
        int extra[kJoinMaxSeg] = {};
        for (int x = 0, lo = 0, hi = k - 1; x < r; ++x) {
            if (x % 2 == 0) extra[lo++] = 1; else extra[hi--] = 1;
        }
        int cut[kJoinMaxSeg + 1];  // segment i = [cut[i], cut[i + 1])
        cut[0] = 0;
        for (int i = 0; i < k; ++i) cut[i + 1] = cut[i] + q + extra[i];
        if (have_stats && n >= k && k >= 2 && set->hist[n] > 0) {
            constexpr float kUnknown = 4.f;  // (bits; 20 equally likely residues would be 4.3)
            float bits[kMaxLen + 1], pre[kMaxLen + 2];
            pre[0] = 0.f;
            for (int p = 0; p < n; ++p) {
                const int back = n - 1 - p;
                float b = p <= back ? (p < kPosStat ? set->pos_bits[0][p] : 0.f) : (back < kPosStat ? set->pos_bits[1][back] : 0.f);
                bits[p] = b > 0.f ? b : kUnknown;
                pre[p + 1] = pre[p] + bits[p];
            }
            auto seg_bits = [&](int b0, int e0) { return pre[e0] - pre[b0]; };
            float def_min = 1e30f;
            for (int i = 0; i < k; ++i) def_min = std::min(def_min, seg_bits(cut[i], cut[i + 1]));
            // best[j][e]: the largest possible minimum over j segments that cover [0, e)
            static thread_local float best[kJoinMaxSeg + 1][kMaxLen + 1];
            static thread_local int8_t from[kJoinMaxSeg + 1][kMaxLen + 1];
            for (int e0 = 1; e0 <= n; ++e0) best[1][e0] = seg_bits(0, e0), from[1][e0] = 0;
            for (int j = 2; j <= k; ++j)
                for (int e0 = j; e0 <= n; ++e0) {
                    float bv = -1.f;
                    int bs = j - 1;
                    for (int s0 = j - 1; s0 < e0; ++s0) {
                        const float v = std::min(best[j - 1][s0], seg_bits(s0, e0));
                        if (v > bv) bv = v, bs = s0;
                    }
                    best[j][e0] = bv;
                    from[j][e0] = (int8_t)bs;
                }
            if (best[k][n] > def_min + 0.75f) {
                int e0 = n;
                for (int j = k; j >= 1; --j) {
                    cut[j] = e0;
                    e0 = from[j][e0];
                }
                cut[0] = 0;
                if (adapted) ++*adapted;
            }
        }
        for (int i = 0; i < k; ++i) tab.seg_start[n][i] = (uint8_t)cut[i];
        for (int i = k; i <= kJoinMaxSeg; ++i) tab.seg_start[n][i] = (uint8_t)n;
    }
    for (int delta = 0; delta <= l_max; ++delta) {
        int np = 0;
        for (int i = 0; i < k; ++i)
            for (int d = -l_max; d <= l_max; ++d)
                if (std::max(std::abs(d), i) + std::abs(d + delta) <= l_max) {
                    if (np >= kJoinMaxProbes) return false;  // (a dropped probe would lose edges)
                    tab.probe_seg[delta][np] = (int8_t)i;
                    tab.probe_shift[delta][np] = (int8_t)d;
                    ++np;
                }
        tab.n_probes[delta] = (int8_t)np;
    }
    return true;
}

// Step A2, host side: the (pattern bucket, text bucket) pairs with len_t - len_p in 0..l_max
// (kPairsAllQuery: 1..l_max; the equal-length pairs belong to the kPairsQueryAll pass).
void schedule_pass(const tcrnet_ctx* ctx, int l_max, int first_check, bool use_join, Schedule::Pass& pass,
                   tcrnet_stats& st) {
    const SeqSet& ps = *pass.pset;
    const SeqSet& ts = *pass.tset;
    // The trie kernel serves the rows whose early exit can act inside the trie (l_max <= kTrieMaxL, the
    // values it is specialised on) and that have at least one text column beyond the trie.
    // (a set loaded for the segment join is bucketed by length only: no trie can be laid over it)
    const bool use_trie = ctx->prefix_trie && first_check > 0 && l_max <= kTrieMaxL && ts.lexicographic;
    for (int m = 1; m < kNumLen; ++m) {
        if (!ps.hist[m]) continue;
        const int n0 = pass.mode == kPairsAllQuery ? m + 1 : m;
        for (int n = n0; n <= std::min(kMaxLen, m + l_max); ++n) {
            if (!ts.hist[n]) continue;
            const int64_t pc = ps.hist[m], tc = ts.hist[n];
            const bool diag = (pass.mode == kPairsSelf || pass.mode == kPairsSelfQuery) && m == n;
            const int64_t pairs = diag ? pc * (pc - 1) / 2 : pc * tc;
            st.pairs_kept += pairs;
            st.cells_kept += pairs * m * n;
            st.columns_kept += pairs * n;
            if (pairs == 0) continue;
            if (use_join && n >= l_max + 1) {  // the text can be cut into l_max + 1 non-empty segments
                std::vector<JoinRow>& jr = pass.join_rows[0];  // (one launch: the word size belongs to the set's plane rows)
                if (jr.empty() || jr.back().m != m) {
                    JoinRow r{};
                    r.m = m;
                    r.p_start = ps.lt.start[m];
                    r.p_count = (int32_t)pc;
                    jr.push_back(r);
                }
                jr.back().t_start[n - m] = ts.lt.start[n];
                jr.back().t_count[n - m] = (int32_t)tc;
                continue;
            }
            const bool trie = use_trie && n > kTrieDepth;
            WorkRow r{};
            r.txt_base = ts.lt.txt_base[n];
            r.p_start = ps.lt.start[m];
            r.p_count = (int32_t)pc;
            r.t_start = ts.lt.start[n];
            r.t_count = (int32_t)tc;
            r.m = m;
            r.n = n;
            r.row_words = ts.lt.row_words[n];
            r.tchunk = trie ? ctx->trie_chunk : ctx->tchunk;
            r.n_tchunks = (int32_t)((tc + r.tchunk - 1) / r.tchunk);
            r.diag = diag ? 1 : 0;
            r.root_begin = ts.trie_root[n];
            r.root_end = ts.trie_root[n + 1];
            pass.part[trie ? 1 : 0][m <= 32 ? 0 : 1].rows.push_back(r);
        }
    }
    for (int trie = 0; trie < 2; ++trie)
        for (Schedule::Part& part : pass.part[trie]) {
            const int tile = trie ? kTrieTile : kTQ;  // patterns per work item
            auto n_items = [tile](const WorkRow& r) { return (int64_t)((r.p_count + tile - 1) / tile) * r.n_tchunks; };
            // big rows first: the small buckets fill the tail of the launch
            std::stable_sort(part.rows.begin(), part.rows.end(), [&](const WorkRow& a, const WorkRow& b) {
                return (long double)a.p_count * a.t_count * a.n > (long double)b.p_count * b.t_count * b.n;
            });
            part.items = 0;
            for (WorkRow& r : part.rows) {
                r.item_begin = part.items;
                part.items += n_items(r);
                part.max_rw = std::max(part.max_rw, (int)r.row_words);
            }
        }
    for (int wide = 0; wide < 2; ++wide) {
        std::vector<JoinRow>& jr = pass.join_rows[wide];
        pass.join_items[wide] = 0;
        for (JoinRow& r : jr) {
            // a work item = 32 patterns x one length difference (0..l_max; empty text buckets return at once)
            r.item_begin = pass.join_items[wide];
            pass.join_items[wide] += (int64_t)((r.p_count + 31) / 32) * (l_max + 1);
        }
    }
}

void make_schedule(const tcrnet_ctx* ctx, int l_max, int first_check, Schedule& sch, tcrnet_stats& st) {
    st.pairs_kept = st.cells_kept = st.columns_kept = st.cells_all = 0;
    {
        long double sum_len = 0, sum_sq = 0;  // sum over unordered pairs of la*lb = ((sum l)^2 - sum l^2) / 2
        for (int l = 1; l < kNumLen; ++l) {
            sum_len += (long double)ctx->row_hist[l] * l;
            sum_sq += (long double)ctx->row_hist[l] * l * l;
        }
        st.cells_all = (int64_t)((sum_len * sum_len - sum_sq) / 2);
    }
    st.pairs_all = ctx->n * (ctx->n - 1) / 2;
    // The join serves the thresholds it is specialised on, with the early exit on (its verification is banded by
    // construction); beyond them the trie / text-chunk kernels.
    const bool can_join = ctx->early_exit && l_max <= kJoinMaxL;
    sch.fast_l1 = can_join && ctx->fast_l1 && l_max <= 1;
    sch.use_join = sch.fast_l1 || (can_join && (ctx->segment_join == 1 ||
                                                (ctx->segment_join < 0 && ctx->prefix_trie)));
    if (ctx->query.loaded) {  // rectangular mode: the pairs with at least one endpoint among the query rows
        const int64_t rest = ctx->n - ctx->query.n;
        st.pairs_all = ctx->query.n * (ctx->query.n - 1) / 2 + ctx->query.n * rest;
        if (sch.use_join) {
            // through the join: ONE pass over all rows as in the all-pairs mode; the emission keeps the pairs that
            // have a query row (kPairsSelfQuery)
            sch.passes.resize(1);
            sch.passes[0].pset = sch.passes[0].tset = &ctx->all;
            sch.passes[0].mode = kPairsSelfQuery;
        } else {
            sch.passes.resize(2);
            sch.passes[0].pset = &ctx->query;
            sch.passes[0].tset = &ctx->all;
            sch.passes[0].mode = kPairsQueryAll;
            sch.passes[1].pset = &ctx->all;
            sch.passes[1].tset = &ctx->query;
            sch.passes[1].mode = kPairsAllQuery;
        }
    } else {
        sch.passes.resize(1);
        sch.passes[0].pset = sch.passes[0].tset = &ctx->all;
        sch.passes[0].mode = kPairsSelf;
    }
    st.work_items = st.work_items_trie = st.work_items_join = 0;
    sch.n_rows = sch.n_join_rows = 0;
    for (Schedule::Pass& pass : sch.passes) {
        schedule_pass(ctx, l_max, first_check, sch.use_join, pass, st);
        for (int trie = 0; trie < 2; ++trie)
            for (int wide = 0; wide < 2; ++wide) {
                st.work_items += pass.part[trie][wide].items;
                if (trie) st.work_items_trie += pass.part[trie][wide].items;
                sch.n_rows += pass.part[trie][wide].rows.size();
            }
        for (int wide = 0; wide < 2; ++wide) {
            st.work_items += pass.join_items[wide];
            st.work_items_join += pass.join_items[wide];
            sch.n_join_rows += pass.join_rows[wide].size();
        }
    }
    st.join_mode = sch.n_join_rows == 0 ? 0 : (l_max <= 1 ? 2 : 1);
}

int upload_schedule(tcrnet_ctx* ctx, const Schedule& sch) {
    TRY(dev_reserve(ctx, ctx->rows, sizeof(WorkRow) * std::max<size_t>(sch.n_rows, 1)));
    WorkRow* dst = (WorkRow*)ctx->rows.p;
    for (const Schedule::Pass& pass : sch.passes)  // same order as run_distance walks them: trie parts first
        for (int trie = 1; trie >= 0; --trie)
            for (int wide = 0; wide < 2; ++wide) {
                const std::vector<WorkRow>& rows = pass.part[trie][wide].rows;
                if (!rows.empty())
                    TRY_CUDA(cudaMemcpyAsync(dst, rows.data(), sizeof(WorkRow) * rows.size(), cudaMemcpyHostToDevice,
                                             ctx->stream));
                dst += rows.size();
            }
    return TCRNET_OK;
}

// (entries of the index of `set` for threshold l_max)
int64_t join_index_entries(const SeqSet& set, int l_max) {
    const int k = l_max + 1;
    int64_t n_idx = 0;
    for (int l = k; l < kNumLen; ++l) n_idx += set.hist[l] * k;
    return n_idx;
}

// The index kernels on stream s (prefix sum in `scan_scratch`, which nothing else may use meanwhile).
int build_join_index(tcrnet_ctx* ctx, int l_max, cudaStream_t s, DevBuf& scan_scratch, int* launches) {
    const SeqSet& set = ctx->all;
    const int64_t n_idx = join_index_entries(set, l_max);
    if (l_max > kJoinMaxL || !make_join_tables(l_max, &set, ctx->join_tab, &ctx->join_adapted)) return TCRNET_ERR_LMAX;
    uint32_t slots = 1024;
    // (one slot per entry at least: a bucket then holds 0.5-1 foreign entries on average, which the walk drops by their
    // segment number / residues; twice the slots cost more in the index build - memset, prefix sum - and in cold
    // directory lines than the shorter lists save: config 5 5.54 -> 5.42 ms, config 4 0.479 -> 0.475 ms)
    while ((int64_t)slots < n_idx && slots < (1u << 30)) slots <<= 1;
    TRY(dev_reserve(ctx, ctx->join_cnt, sizeof(uint32_t) * (size_t)slots));
    TRY(dev_reserve(ctx, ctx->join_dir, sizeof(uint32_t) * ((size_t)slots + 1)));
    TRY(dev_reserve(ctx, ctx->join_entries, sizeof(uint2) * (size_t)std::max<int64_t>(n_idx, 1)));
    TRY(dev_reserve(ctx, scan_scratch, scan_scratch_bytes((int64_t)slots)));
    TRY_CUDA(cudaMemsetAsync(ctx->join_cnt.p, 0, sizeof(uint32_t) * (size_t)slots, s));
    TRY_CUDA(launch_join_index(set.planes.p, set.wide_planes, set.lt, set.n, ctx->join_tab,
                               (uint32_t*)ctx->join_cnt.p, (uint32_t*)ctx->join_dir.p, (uint2*)ctx->join_entries.p, slots,
                               scan_scratch.p, s, launches));
    ctx->join_slots = slots;
    ctx->join_l_max = l_max;
    return TCRNET_OK;
}

// Whatever the load left running on the second stream (the index built ahead, below) is ordered before the main
// stream's next operation.
int settle_index(tcrnet_ctx* ctx) {
    if (ctx->index_pending) {
        TRY_CUDA(cudaStreamWaitEvent(ctx->stream, ctx->ev_index, 0));
        ctx->index_pending = false;
    }
    return TCRNET_OK;
}

// Built AHEAD: a load ends with a host synchronisation and the build that follows starts with host work (schedule,
// reservations); the index depends on the load and on l_max alone, so the load starts building it on the second stream
// for the threshold of the previous build (the usual case: the same threshold again) and returns without waiting.
// A build at another threshold waits for it and builds its own.
int build_join_index_ahead(tcrnet_ctx* ctx, int* launches) {
    const int l_max = ctx->ahead_l_max;
    const bool join_on = ctx->early_exit && ctx->segment_join != 0;  // (ahead_l_max: a build did use the join)
    // (timing level 2 measures the phases one after the other: nothing is built ahead there)
    if (l_max < 0 || l_max > kJoinMaxL || !join_on || ctx->timing >= 2) return TCRNET_OK;
    if (join_index_entries(ctx->all, l_max) == 0) return TCRNET_OK;
    TRY(build_join_index(ctx, l_max, ctx->side_stream, ctx->join_scan_scratch, launches));
    TRY_CUDA(cudaEventRecord(ctx->ev_index, ctx->side_stream));
    ctx->index_pending = true;
    return TCRNET_OK;
}

// Segment index of the texts of ctx->all for threshold l_max (kept until the next load / another threshold).
int ensure_join_index(tcrnet_ctx* ctx, int l_max, int* launches) {
    tcrnet_stats& st = ctx->stats;
    st.ms_index = 0.f;
    st.join_index_entries = join_index_entries(ctx->all, l_max);
    TRY(settle_index(ctx));
    struct SetAdapted {  // (whichever path leaves the index in place: the count belongs to it)
        tcrnet_ctx* c;
        ~SetAdapted() { c->stats.join_adapted_lengths = c->join_adapted; }
    } set_adapted{ctx};
    ctx->ahead_l_max = l_max;
    if (ctx->join_l_max == l_max) return TCRNET_OK;
    TRY_CUDA(rec(ctx, 6, 2));
    TRY(build_join_index(ctx, l_max, ctx->stream, ctx->scan_scratch, launches));
    TRY_CUDA(rec(ctx, 7, 2));
    if (ctx->timing >= 2) st.ms_index = -1.f;  // measured once the events have completed (distance_phase)
    return TCRNET_OK;
}

// cap: capacity of keys_a (the pairs the distance kernels record); cap_b: of keys_b (grouped loads only: the edges
// between rows after the expansion).
// expand_only: the recorded pairs in keys_a are complete, only keys_b was too small - redo the expansion alone.
// The counters and per-row counts a distance pass starts from (issued ahead of the index kernels for the first pass,
// so that no memset sits between two kernels of the chain index -> join -> expansion).
int reset_build_counters(tcrnet_ctx* ctx, bool expand_only) {
    cudaStream_t s = ctx->stream;
    HostCtrl* dc = d_ctrl(ctx);
    static_assert(offsetof(HostCtrl, queue) == offsetof(HostCtrl, edge_count) + 9 * sizeof(unsigned long long), "one memset");
    static_assert(offsetof(HostCtrl, edge_total) == offsetof(HostCtrl, queue) + kTrieQueues * sizeof(unsigned long long), "one memset");
    static_assert(offsetof(HostCtrl, cand_count) == offsetof(HostCtrl, edge_total) + sizeof(unsigned long long), "one memset");
    static_assert(offsetof(HostCtrl, n_huge) == offsetof(HostCtrl, cand_count) + sizeof(unsigned long long), "one memset");
    if (expand_only) {
        TRY_CUDA(cudaMemsetAsync(&dc->edge_total, 0, sizeof(unsigned long long), s));
        TRY_CUDA(cudaMemsetAsync(&dc->n_huge, 0, sizeof(unsigned long long), s));
    } else {  // edge_count, work[8], queue[], edge_total, cand_count, n_huge
        TRY_CUDA(cudaMemsetAsync(&dc->edge_count, 0, sizeof(unsigned long long) * (12 + kTrieQueues), s));
    }
    TRY_CUDA(cudaMemsetAsync(ctx->row_count.p, 0, sizeof(int32_t) * (size_t)ctx->n, s));
    TRY_CUDA(cudaMemsetAsync(ctx->deg.p, 0, sizeof(int32_t) * (size_t)ctx->n, s));
    return TCRNET_OK;
}

int assemble_reserve(tcrnet_ctx* ctx, int64_t bound);
int assemble_launch(tcrnet_ctx* ctx, const unsigned long long* edges, unsigned long long* bucket,
                    const unsigned long long* n_dev, int64_t bound, bool distinct_keys, int* launches);
int assemble_finish(tcrnet_ctx* ctx, int64_t n_keys, const unsigned long long* bucket, int* launches);

// assemble_too: step A6 is launched right behind the distance kernels, on the edge count as the device holds it, and
// the ONE synchronisation at the end serves both (the host then finds out whether the buffers were large enough).
int run_distance(tcrnet_ctx* ctx, const Schedule& sch, int l_max, int first_check, uint64_t cap, uint64_t cap_b, int shard,
                 int n_shards, bool expand_only, bool counters_cleared, int* launches, bool assemble_too = false) {
    cudaStream_t s = ctx->stream;
    HostCtrl* dc = d_ctrl(ctx);
    static_assert(offsetof(HostCtrl, queue) == offsetof(HostCtrl, edge_count) + 9 * sizeof(unsigned long long), "one memset");
    static_assert(offsetof(HostCtrl, edge_total) == offsetof(HostCtrl, queue) + kTrieQueues * sizeof(unsigned long long), "one memset");
    static_assert(offsetof(HostCtrl, cand_count) == offsetof(HostCtrl, edge_total) + sizeof(unsigned long long), "one memset");
    if (!counters_cleared) TRY(reset_build_counters(ctx, expand_only));
    int n_queues = 0;
    const WorkRow* d_rows = (const WorkRow*)ctx->rows.p;
    if (!expand_only) TRY_CUDA(rec(ctx, 4, 1));
    for (const Schedule::Pass& pass : sch.passes) {
        if (expand_only) break;
        DistanceParams p{};
        p.l_max = l_max;
        p.mode = pass.mode;
        p.n_query = (int32_t)ctx->query.n;
        p.shard = shard;
        p.n_shards = n_shards;
        p.pat_stride = pass.pset->pat_stride;
        p.pat = (const uint8_t*)pass.pset->pat.p;
        p.perm_p = (const int32_t*)pass.pset->perm.p;
        p.txt = (const uint32_t*)pass.tset->txt.p;
        p.perm_t = (const int32_t*)pass.tset->perm.p;
        for (int k = 0; k <= kTrieDepth; ++k) p.trie[k] = pass.tset->trie_levels.p[k];
        p.edges = (unsigned long long*)ctx->keys_a.p;
        p.row_count = (int32_t*)ctx->row_count.p;
        p.deg = (int32_t*)ctx->deg.p;
        p.group_start = ctx->all.grouped ? (const uint32_t*)ctx->all.group_start.p : nullptr;
        p.members = ctx->all.grouped ? (const int32_t*)ctx->all.members.p : nullptr;
        p.edge_count = &dc->edge_count;
        p.edge_cap = cap;
        p.work = dc->work;
        for (int trie = 1; trie >= 0; --trie)
            for (int wide = 0; wide < 2; ++wide) {
                const Schedule::Part& part = pass.part[trie][wide];
                if (!part.rows.empty()) {
                    p.rows = d_rows;
                    p.n_rows = (int32_t)part.rows.size();
                    if (trie) {
                        if (n_queues >= kTrieQueues) return TCRNET_ERR_STATE;  // at most 2 passes x 2 word sizes
                        p.queue = dc->queue + n_queues++;
                        p.n_items = part.items;
                        TRY_CUDA(launch_distance_trie(p, part.items, wide != 0, ctx->count_work != 0, ctx->n_sm, s, launches));
                    } else
                        TRY_CUDA(launch_distance(p, part.items, wide != 0, first_check, ctx->count_work != 0,
                                                 part.max_rw, s, launches));
                }
                d_rows += part.rows.size();
            }
        for (int wide = 0; wide < 2; ++wide) {
            const std::vector<JoinRow>& jr = pass.join_rows[wide];
            if (!jr.empty()) {
                p.n_items = pass.join_items[wide];
                JoinIndex index{(const uint32_t*)ctx->join_dir.p, (const uint2*)ctx->join_entries.p, ctx->join_slots - 1u};
                TRY_CUDA(launch_join(p, jr.data(), (int)jr.size(), pass.pset->planes.p, pass.pset->wide_planes, index,
                                     ctx->join_tab, (uint2*)ctx->join_cand.p,
                                     (uint8_t*)ctx->join_cand.p + sizeof(uint2) * (size_t)ctx->join_cand_cap, &dc->cand_count,
                                     (unsigned long long)ctx->join_cand_cap, ctx->count_work != 0, ctx->n_sm, s, launches));
            }
        }
    }
    if (!expand_only) TRY_CUDA(rec(ctx, 5, 1));
    if (ctx->all.grouped) {
        // The rows of every shared sequence are joined to each other (k_emit_cliques) on the second stream, beside the
        // expansion below: the two are independent (they share the cursor of keys_b and the per-row counters, both
        // updated atomically).  Beside the join kernel - where it ran before - it cost the same step time but shared
        // the SMs with the kernel the roofline is reported for (81 us instead of 62 us at config 4).
        TRY_CUDA(cudaEventRecord(ctx->ev_fork, s));
        TRY_CUDA(cudaStreamWaitEvent(ctx->side_stream, ctx->ev_fork, 0));
        TRY_CUDA(launch_emit_cliques((const int32_t*)ctx->all.members.p, (const int32_t*)ctx->all.uid_of.p,
                                     (const uint32_t*)ctx->all.group_start.p, ctx->n, (unsigned long long*)ctx->keys_b.p,
                                     &dc->edge_total, cap_b, (int32_t*)ctx->row_count.p, (int32_t*)ctx->deg.p, shard, n_shards,
                                     ctx->side_stream, launches));
        TRY_CUDA(cudaEventRecord(ctx->ev_join, ctx->side_stream));
        // the recorded pairs of distinct sequences -> edges between rows (keys_b), counted for the CSR step
        const uint32_t* gs = (const uint32_t*)ctx->all.group_start.p;
        const int32_t* mem = (const int32_t*)ctx->all.members.p;
        TRY_CUDA(launch_expand_entries((const unsigned long long*)ctx->keys_a.p, &dc->edge_count, cap, gs, mem,
                                       (unsigned long long*)ctx->keys_b.p, &dc->edge_total, cap_b, (int32_t*)ctx->row_count.p,
                                       (int32_t*)ctx->deg.p, ctx->expand_huge.p, &dc->n_huge, kExpandHugeCap,
                                       /*huge_possible=*/ctx->max_group > 64u, ctx->n_sm, s, launches));
        TRY_CUDA(cudaStreamWaitEvent(s, ctx->ev_join, 0));  // the cliques are in
        TRY_CUDA(cudaMemcpyAsync(&ctx->h_ctrl->edge_total, &dc->edge_total, sizeof(unsigned long long), cudaMemcpyDeviceToHost, s));
    }
    TRY_CUDA(cudaMemcpyAsync(&ctx->h_ctrl->edge_count, &dc->edge_count, sizeof(unsigned long long) * 9,
                             cudaMemcpyDeviceToHost, s));
    TRY_CUDA(cudaMemcpyAsync(&ctx->h_ctrl->cand_count, &dc->cand_count, sizeof(unsigned long long), cudaMemcpyDeviceToHost, s));
    if (assemble_too) {
        const bool grouped = ctx->all.grouped;  // (grouped: the edges are in keys_b and keys_a is free again)
        TRY(assemble_launch(ctx, (const unsigned long long*)(grouped ? ctx->keys_b.p : ctx->keys_a.p),
                            (unsigned long long*)(grouped ? ctx->keys_a.p : ctx->keys_b.p),
                            grouped ? &dc->edge_total : &dc->edge_count, (int64_t)(grouped ? cap_b : cap), true, launches));
    }
    TRY_CUDA(cudaStreamSynchronize(s));
    return TCRNET_OK;
}

// Steps A2-A5 for the work items of one shard: unsorted keys in keys_a, ctx->n_keys of them.
int distance_phase(tcrnet_ctx* ctx, int l_max, int shard, int n_shards, int* launches, bool assemble_too = false) {
    ctx->assembled = false;
    assemble_too = assemble_too && ctx->timing < 2;  // (level 2 times the phases one after the other)
    tcrnet_stats& st = ctx->stats;
    const int64_t n = ctx->n;
    int first_check = 0;
    if (ctx->early_exit) {
        first_check = ctx->first_check_opt ? ctx->first_check_opt : l_max + 2;
        first_check = std::max(3, std::min(8, first_check));
    }
    st.first_check = first_check;
    st.l_max = l_max;
    // identical rows are joined for every l_max: if those edges alone exceed the limit, fail before any work
    // (one sequence repeated g times means g (g - 1) / 2 of them)
    if (ctx->all.grouped && ctx->clique_edges > ctx->edge_limit) return TCRNET_ERR_EDGE_OVERFLOW;
    Schedule sch;
    make_schedule(ctx, l_max, first_check, sch, st);
    TRY_CUDA(rec(ctx, 0, 2));
    TRY(upload_schedule(ctx, sch));
    // distances + emission (second pass only if the edge buffer was too small)
    int64_t cap = ctx->edge_capacity_opt > 0 ? ctx->edge_capacity_opt : std::max<int64_t>((int64_t)1 << 20, 16 * n);
    cap = std::min(cap, ctx->edge_limit);
    cap = std::max<int64_t>(cap, 1);
    if (ctx->keys_a.p && (int64_t)(ctx->keys_a.bytes / 8) > cap) cap = std::min<int64_t>(ctx->keys_a.bytes / 8, ctx->edge_limit);
    TRY(dev_reserve(ctx, ctx->keys_a, sizeof(unsigned long long) * (size_t)cap));
    TRY(dev_reserve(ctx, ctx->row_count, sizeof(int32_t) * (size_t)n));
    TRY(dev_reserve(ctx, ctx->deg, sizeof(int32_t) * (size_t)n));
    const bool grouped = ctx->all.grouped;
    int64_t cap_b = 0;
    if (grouped) TRY(dev_reserve(ctx, ctx->expand_huge, 16 * (size_t)kExpandHugeCap));
    if (grouped) {
        cap_b = std::max<int64_t>(cap, (int64_t)(ctx->keys_b.bytes / 8));
        cap_b = std::min(cap_b, ctx->edge_limit);
        TRY(dev_reserve(ctx, ctx->keys_b, sizeof(unsigned long long) * (size_t)cap_b));
    }
    if (assemble_too) {
        // every buffer of step A6 by its upper bound, before anything is launched; the scratch of the scatter is the
        // other key buffer (grouped: keys_a, free once the expansion has read the recorded pairs)
        if (grouped && cap_b > cap) {
            cap = cap_b;
            TRY(dev_reserve(ctx, ctx->keys_a, sizeof(unsigned long long) * (size_t)cap));
        }
        if (!grouped) TRY(dev_reserve(ctx, ctx->keys_b, sizeof(unsigned long long) * (size_t)cap));
        TRY(assemble_reserve(ctx, grouped ? cap_b : cap));
    }
    // the first pass's resets go ahead of the index kernels: index -> join -> cliques -> expansion is one chain of kernels
    TRY(reset_build_counters(ctx, false));
    bool counters_cleared = true;
    st.ms_index = 0.f;
    st.join_index_entries = 0;
    if (sch.n_join_rows) {
        TRY(ensure_join_index(ctx, l_max, launches));
        if (l_max >= 2 && ctx->join_cand_cap == 0) {
            // queue of the pairs that pass the filters: 8 + 1 bytes each (grown to the exact count if too small)
            ctx->join_cand_cap = std::max<int64_t>((int64_t)1 << 20, 8 * ctx->all.n);
            TRY(dev_reserve(ctx, ctx->join_cand, 9 * (size_t)ctx->join_cand_cap));
        }
    }
    if (sch.n_rows) {  // the prefix-trie / text-chunk kernels run: they read txt (and the trie)
        for (Schedule::Pass& pass : sch.passes) {
            TRY(ensure_text_tables(ctx, const_cast<SeqSet&>(*pass.pset), launches));
            TRY(ensure_text_tables(ctx, const_cast<SeqSet&>(*pass.tset), launches));
        }
        // the rows were laid out before the trie roots were known
        sch = Schedule();
        make_schedule(ctx, l_max, first_check, sch, st);
        TRY(upload_schedule(ctx, sch));
    }
    st.trie_nodes = ctx->all.trie_nodes;

    int64_t n_keys = 0;
    st.distance_passes = 0;
    for (bool expand_only = false;;) {
        if (!expand_only) ++st.distance_passes;
        const bool with_a6 = assemble_too && st.distance_passes == 1 && !expand_only;  // (the first pass only)
        TRY(run_distance(ctx, sch, l_max, first_check, (uint64_t)cap, (uint64_t)cap_b, shard, n_shards, expand_only,
                         counters_cleared, launches, with_a6));
        counters_cleared = false;
        const int64_t n_rec = (int64_t)ctx->h_ctrl->edge_count;  // pairs recorded by the distance kernels
        const int64_t n_cand = (int64_t)ctx->h_ctrl->cand_count;
        if (!expand_only && n_cand > ctx->join_cand_cap) {
            // the verification queue of the join was too small: grow it to the exact count and run again
            if (st.distance_passes >= 3) return TCRNET_ERR_CUDA;  // cannot happen: same input
            ctx->join_cand_cap = n_cand;
            TRY(dev_reserve(ctx, ctx->join_cand, 9 * (size_t)n_cand));
            continue;
        }
        n_keys = grouped ? (int64_t)ctx->h_ctrl->edge_total : n_rec;
        if (n_rec > ctx->edge_limit || (n_rec <= cap && n_keys > ctx->edge_limit)) return TCRNET_ERR_EDGE_OVERFLOW;
        if (n_rec > cap) {  // the record buffer was too small: grow it to the exact count and run again
            if (st.distance_passes >= 3) return TCRNET_ERR_CUDA;  // cannot happen: same input
            cap = n_rec;
            TRY(dev_reserve(ctx, ctx->keys_a, sizeof(unsigned long long) * (size_t)cap));
            continue;
        }
        if (!grouped || n_keys <= cap_b) {
            ctx->assembled = with_a6;  // (every count fits: what step A6 was launched on is the whole edge list)
            break;
        }
        if (expand_only) return TCRNET_ERR_CUDA;  // cannot happen: exact size
        cap_b = n_keys;
        TRY(dev_reserve(ctx, ctx->keys_b, sizeof(unsigned long long) * (size_t)cap_b));
        expand_only = true;
    }
    if (grouped) std::swap(ctx->keys_a, ctx->keys_b);  // the edges between rows are what the CSR step takes
    // (... and has taken already if it was launched with the first pass: its scratch is then in keys_b)
    st.ms_kernel = 0.f;
    // (of the last pass; both events complete: synchronised above)
    if (ctx->timing >= 1) TRY_CUDA(cudaEventElapsedTime(&st.ms_kernel, ctx->ev[4], ctx->ev[5]));
    st.lane_columns_exec = (int64_t)ctx->h_ctrl->work[0];
    st.lane_tests_exec = (int64_t)ctx->h_ctrl->work[1];
    st.lane_pairs_exec = (int64_t)ctx->h_ctrl->work[2];
    st.lane_prefix_tests_exec = (int64_t)ctx->h_ctrl->work[3];
    st.lane_columns_live = (int64_t)ctx->h_ctrl->work[4];
    st.join_probes = (int64_t)ctx->h_ctrl->work[5];
    st.join_entries = (int64_t)ctx->h_ctrl->work[6];
    st.join_candidates = (int64_t)ctx->h_ctrl->work[7];
    st.join_survivors = st.join_mode ? (int64_t)ctx->h_ctrl->work[4] : 0;
    st.join_diagonals = st.join_verified_edges = 0;
    if (st.join_mode && st.work_items == st.work_items_join) {  // (the counters are shared with the other kernels)
        st.join_diagonals = (int64_t)ctx->h_ctrl->work[0];
        st.join_verified_edges = (int64_t)ctx->h_ctrl->work[3];
        st.lane_columns_exec = st.lane_prefix_tests_exec = st.lane_columns_live = 0;
    }
    if (st.ms_index < 0.f) TRY_CUDA(cudaEventElapsedTime(&st.ms_index, ctx->ev[6], ctx->ev[7]));
    TRY_CUDA(rec(ctx, 1, 2));
    ctx->n_keys = n_keys;
    return TCRNET_OK;
}

// Buffers of step A6 for n rows and up to `bound` keys (no-ops when they are large enough).
int assemble_reserve(tcrnet_ctx* ctx, int64_t bound) {
    const int64_t n = ctx->n;
    TRY(dev_reserve(ctx, ctx->row_count, sizeof(int32_t) * (size_t)n));
    TRY(dev_reserve(ctx, ctx->long_rows, sizeof(int32_t) * (size_t)n));
    TRY(dev_reserve(ctx, ctx->scan_scratch, scan_scratch_bytes(n)));
    TRY(dev_reserve(ctx, ctx->row_ptr, sizeof(int64_t) * (size_t)(n + 1)));
    TRY(dev_reserve(ctx, ctx->col, sizeof(int32_t) * (size_t)std::max<int64_t>(bound, 1)));
    TRY(dev_reserve(ctx, ctx->deg, sizeof(int32_t) * (size_t)n));
    return TCRNET_OK;
}

// The kernels of step A6 on the keys in `edges` (their number: `bound`, or *n_dev with `bound` the capacity of edges,
// bucket and col - launch_csr_unsorted), per-row counts in row_count / deg; the count of the long rows is on its way to
// the host.  Nothing is synchronised.
int assemble_launch(tcrnet_ctx* ctx, const unsigned long long* edges, unsigned long long* bucket,
                    const unsigned long long* n_dev, int64_t bound, bool distinct_keys, int* launches) {
    cudaStream_t s = ctx->stream;
    HostCtrl* dc = d_ctrl(ctx);
    TRY_CUDA(rec(ctx, 2, 2));
    TRY_CUDA(launch_csr_unsorted(edges, n_dev, bound, ctx->n, (int32_t*)ctx->row_count.p, (int64_t*)ctx->row_ptr.p, bucket,
                                 (int32_t*)ctx->col.p, (int32_t*)ctx->deg.p, (int32_t*)ctx->long_rows.p, &dc->n_long,
                                 ctx->scan_scratch.p, distinct_keys, s, launches));
    TRY_CUDA(cudaMemcpyAsync(&ctx->h_ctrl->n_long, &dc->n_long, sizeof(uint32_t), cudaMemcpyDeviceToHost, s));
    return TCRNET_OK;
}

int assemble_sort_long(tcrnet_ctx* ctx, const unsigned long long* bucket, int* launches) {
    return launch_sort_long_rows(ctx->n, (const int64_t*)ctx->row_ptr.p, bucket, (int32_t*)ctx->col.p,
                                 (const int32_t*)ctx->long_rows.p, &d_ctrl(ctx)->n_long, ctx->stream, launches) == cudaSuccess
               ? TCRNET_OK : TCRNET_ERR_CUDA;
}

// ... once the stream has been synchronised behind assemble_launch: the rows of more than 256 neighbours (if any: they
// are ordered by a kernel of their own), bookkeeping.
int assemble_finish(tcrnet_ctx* ctx, int64_t n_keys, const unsigned long long* bucket, int* launches) {
    tcrnet_stats& st = ctx->stats;
    if (ctx->timing < 2 && n_keys > 0 && ctx->h_ctrl->n_long > 0) {
        TRY(assemble_sort_long(ctx, bucket, launches));
        TRY_CUDA(cudaStreamSynchronize(ctx->stream));
    }
    st.ms_sort = st.ms_csr = 0.f;
    if (ctx->timing >= 2) {
        TRY_CUDA(cudaEventElapsedTime(&st.ms_sort, ctx->ev[1], ctx->ev[2]));
        TRY_CUDA(cudaEventElapsedTime(&st.ms_csr, ctx->ev[2], ctx->ev[3]));
    }
    st.n_edges = n_keys;
    ctx->n_edges = n_keys;
    ctx->have_keys = false;
    ctx->have_dist = false;
    drop_observables(ctx);
    ctx->built = true;
    return TCRNET_OK;
}

// Step A6 on the n_keys unsorted keys (u << 32) | v in keys_a: per-row counts (left in row_count by the emission
// when counts_ready), prefix sum -> row_ptr, every edge into a slot of its row, rows ordered; degrees.
int assemble_phase(tcrnet_ctx* ctx, int64_t n_keys, bool counts_ready, int* launches) {
    cudaStream_t s = ctx->stream;
    const int64_t n = ctx->n;
    TRY(assemble_reserve(ctx, n_keys));
    TRY(dev_reserve(ctx, ctx->keys_b, sizeof(unsigned long long) * (size_t)std::max<int64_t>(n_keys, 1)));
    if (!counts_ready) {
        TRY_CUDA(cudaMemsetAsync(ctx->row_count.p, 0, sizeof(int32_t) * (size_t)n, s));
        TRY_CUDA(cudaMemsetAsync(ctx->deg.p, 0, sizeof(int32_t) * (size_t)n, s));
        TRY_CUDA(launch_count_rows((const unsigned long long*)ctx->keys_a.p, n_keys, (int32_t*)ctx->row_count.p,
                                   (int32_t*)ctx->deg.p, s, launches));
    }
    unsigned long long* bucket = (unsigned long long*)ctx->keys_b.p;
    TRY(assemble_launch(ctx, (const unsigned long long*)ctx->keys_a.p, bucket, nullptr, n_keys, counts_ready, launches));
    if (ctx->timing >= 2) {  // (the phase events bracket the whole step: no read-back in between)
        if (n_keys > 0) TRY(assemble_sort_long(ctx, bucket, launches));
        TRY_CUDA(rec(ctx, 3, 2));
    }
    TRY_CUDA(cudaStreamSynchronize(s));
    return assemble_finish(ctx, n_keys, bucket, launches);
}

// Distance labels of the current CSR's edges (labels.cu), computed on first use.
int ensure_edge_distances(tcrnet_ctx* ctx, int* launches) {
    if (ctx->have_dist) return TCRNET_OK;
    cudaStream_t s = ctx->stream;
    TRY(dev_reserve(ctx, ctx->inv_perm, sizeof(int32_t) * (size_t)ctx->n));
    TRY(dev_reserve(ctx, ctx->edge_dist, (size_t)std::max<int64_t>(ctx->n_edges, 1)));
    if (ctx->all.grouped)
        TRY_CUDA(launch_inverse_perm_groups((const int32_t*)ctx->all.perm.p, ctx->all.n, (const uint32_t*)ctx->all.group_start.p,
                                            (const int32_t*)ctx->all.members.p, (int32_t*)ctx->inv_perm.p, s, launches));
    else
        TRY_CUDA(launch_inverse_perm((const int32_t*)ctx->all.perm.p, ctx->n, (int32_t*)ctx->inv_perm.p, s, launches));
    TRY(dev_reserve(ctx, ctx->edge_row, sizeof(int32_t) * (size_t)std::max<int64_t>(ctx->n_edges, 1)));
    TRY_CUDA(launch_edge_rows((const int64_t*)ctx->row_ptr.p, ctx->n, (int32_t*)ctx->edge_row.p, s, launches));
    TRY_CUDA(launch_edge_distances((const int32_t*)ctx->edge_row.p, (const int32_t*)ctx->col.p, ctx->n_edges,
                                   (const int32_t*)ctx->inv_perm.p, ctx->all.planes.p, ctx->all.wide_planes,
                                   (uint8_t*)ctx->edge_dist.p, s, launches));
    ctx->have_dist = true;
    return TCRNET_OK;
}

}  // namespace

extern "C" {

// (visibility comes from the TCRNET_API declarations in tcrnet.h)
int tcrnet_version(void) { return TCRNET_VERSION; }

const char* tcrnet_strerror(int status) {
    switch (status) {
        case TCRNET_OK: return "ok";
        case TCRNET_ERR_ARG: return "invalid argument";
        case TCRNET_ERR_LENGTH: return "sequence length outside 1..64";
        case TCRNET_ERR_RESIDUE: return "residue byte outside 'A'..'Z'";
        case TCRNET_ERR_LMAX: return "l_max outside 0..64";
        case TCRNET_ERR_STATE: return "call out of order (load before build, build before csr/degrees)";
        case TCRNET_ERR_NOMEM: return "out of device memory";
        case TCRNET_ERR_EDGE_OVERFLOW: return "edge count exceeds the configured limit";
        case TCRNET_ERR_CUDA: return "CUDA runtime error";
        case TCRNET_ERR_CAPACITY: return "size beyond the fixed capacity of a no-allocation call";
        default: return "unknown status";
    }
}

int tcrnet_create(tcrnet_ctx** out, int device, void* cuda_stream, const tcrnet_allocator* allocator) {
    if (!out) return TCRNET_ERR_ARG;
    *out = nullptr;
    if (allocator && (!allocator->alloc || !allocator->free)) return TCRNET_ERR_ARG;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) {
        (void)cudaGetLastError();
        return TCRNET_ERR_CUDA;
    }
    tcrnet_ctx* ctx = new (std::nothrow) tcrnet_ctx();
    if (!ctx) return TCRNET_ERR_NOMEM;
    ctx->device = device;
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    if (allocator) {
        ctx->alloc = *allocator;
        ctx->has_alloc = true;
    }
    cudaError_t e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->n_sm, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) e = cudaMallocHost((void**)&ctx->h_ctrl, sizeof(HostCtrl));
    for (int i = 0; e == cudaSuccess && i < 8; ++i) e = cudaEventCreate(&ctx->ev[i]);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->side_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_index, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        tcrnet_destroy(ctx);
        return TCRNET_ERR_CUDA;
    }
    if (dev_reserve(ctx, ctx->ctrl, sizeof(HostCtrl)) != TCRNET_OK) {
        tcrnet_destroy(ctx);
        return TCRNET_ERR_NOMEM;
    }
    *out = ctx;
    return TCRNET_OK;
}

void tcrnet_destroy(tcrnet_ctx* ctx) {
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    if (ctx->side_stream) {
        cudaStreamSynchronize(ctx->side_stream);
        cudaStreamDestroy(ctx->side_stream);
    }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
    if (ctx->ev_index) cudaEventDestroy(ctx->ev_index);
    DevBuf* bufs[] = {
        &ctx->all.perm, &ctx->all.pat, &ctx->all.txt, &ctx->all.trie, &ctx->query.perm, &ctx->query.pat,
        &ctx->query.txt, &ctx->query.trie, &ctx->all.planes, &ctx->query.planes, &ctx->join_cand, &ctx->expand_huge,
        &ctx->join_scan_scratch, &ctx->join_cnt, &ctx->join_dir, &ctx->join_entries, &ctx->join_rows, &ctx->inv_perm,
        &ctx->edge_row, &ctx->edge_dist, &ctx->edge_dist_b, &ctx->flags, &ctx->flag_pos, &ctx->in_res, &ctx->in_len,
        &ctx->offsets, &ctx->perm_tmp, &ctx->trie_scratch, &ctx->keys_a, &ctx->keys_b, &ctx->radix_scratch,
        &ctx->scan_scratch, &ctx->rows, &ctx->row_ptr, &ctx->col, &ctx->row_count, &ctx->long_rows,
        &ctx->all.group_start, &ctx->all.members, &ctx->all.uid_of, &ctx->dd_table, &ctx->dd_hash, &ctx->dd_rep,
        &ctx->dd_first, &ctx->dd_rank, &ctx->dd_count, &ctx->dd_len, &ctx->dd_off, &ctx->dd_offsets, &ctx->deg,
        &ctx->ctrl, &ctx->obs_ctrl, &ctx->deg_hist, &ctx->nn_sum, &ctx->class_sum, &ctx->knn, &ctx->cc_parent,
        &ctx->cc_count, &ctx->cc_label, &ctx->cc_size, &ctx->perc_rank, &ctx->perc_seen, &ctx->perc_deg,
        &ctx->perc_hist, &ctx->perc_lcc};
    for (DevBuf* b : bufs) dev_free(ctx, *b);
    if (ctx->h_ctrl) cudaFreeHost(ctx->h_ctrl);
    for (cudaEvent_t ev : ctx->ev)
        if (ev) cudaEventDestroy(ev);
    (void)cudaGetLastError();
    delete ctx;
}

int tcrnet_load_device(tcrnet_ctx* ctx, const uint8_t* residues_dev, const int32_t* lengths_dev, int64_t n,
                       int64_t total_len) {
    if (!ctx || !residues_dev || !lengths_dev || n < 1 || n > 0x7ffffffeLL || total_len < n) return TCRNET_ERR_ARG;
    TRY_CUDA(cudaSetDevice(ctx->device));
    TRY(settle_index(ctx));  // (an index still being built ahead reads the tables this load rewrites)
    drop_load(ctx);
    int launches = 0;
    TRY_CUDA(rec(ctx, 0, 2));
    TRY(load_from_device(ctx, residues_dev, lengths_dev, n, total_len, &launches));  // (ends synchronised)
    ctx->stats.ms_load = 0.f;
    if (ctx->timing >= 2) {
        TRY_CUDA(cudaEventRecord(ctx->ev[1], ctx->stream));
        TRY_CUDA(cudaEventSynchronize(ctx->ev[1]));
        TRY_CUDA(cudaEventElapsedTime(&ctx->stats.ms_load, ctx->ev[0], ctx->ev[1]));
    }
    ctx->stats.launches_load = launches;
    return TCRNET_OK;
}

int tcrnet_load(tcrnet_ctx* ctx, const uint8_t* residues, const int32_t* lengths, int64_t n) {
    return tcrnet_load_sized(ctx, residues, INT64_MAX, lengths, n);
}

int tcrnet_load_sized(tcrnet_ctx* ctx, const uint8_t* residues, int64_t residues_size, const int32_t* lengths,
                      int64_t n) {
    if (!ctx || !residues || !lengths || n < 1 || n > 0x7ffffffeLL || residues_size < n) return TCRNET_ERR_ARG;
    TRY_CUDA(cudaSetDevice(ctx->device));
    TRY(settle_index(ctx));
    drop_load(ctx);
    // The lengths go first.  The residue array is sized by their sum, which only a host pass over them gives: that pass
    // runs in blocks of rows and, as long as the buffer of the previous load is large enough, the residues of every
    // finished block are copied at once - the pass hides behind the copies instead of preceding them (config 4: 0.25 ms
    // of a 0.9 ms load).  Validation proper happens on the device; this pass only keeps the sum meaningful.
    DevBuf& d_res = ctx->in_res;
    DevBuf& d_len = ctx->in_len;
    cudaStream_t s = ctx->stream;
    int rc = dev_reserve(ctx, d_len, sizeof(int32_t) * (size_t)n);
    if (rc != TCRNET_OK) return rc;
    TRY_CUDA(rec(ctx, 0, 2));
    TRY_CUDA(cudaMemcpyAsync(d_len.p, lengths, sizeof(int32_t) * (size_t)n, cudaMemcpyHostToDevice, s));
    constexpr int64_t kBlockRows = 1 << 16, kInner = 4096;  // (4096 x kMaxLen fits 32 bits: the inner sums vectorise)
    int64_t total_len = 0, copied = 0;
    uint32_t bad = 0;
    bool too_short = false;
    cudaError_t ce = cudaSuccess;
    for (int64_t b0 = 0; b0 < n && !bad && !too_short && ce == cudaSuccess; b0 += kBlockRows) {
        const int64_t b1 = std::min<int64_t>(n, b0 + kBlockRows);
        for (int64_t i0 = b0; i0 < b1; i0 += kInner) {
            const int64_t i1 = std::min<int64_t>(b1, i0 + kInner);
            uint32_t sum = 0, any = 0;
            for (int64_t i = i0; i < i1; ++i) {
                const uint32_t l = (uint32_t)lengths[i];
                sum += l;
                any |= l - 1u;
            }
            bad |= any & ~(uint32_t)(kMaxLen - 1);  // some l - 1 >= kMaxLen (kMaxLen is a power of two)
            total_len += sum;
        }
        too_short = !bad && total_len > residues_size;  // (checked before a byte of the block is read)
        if (!bad && !too_short && d_res.p && (size_t)total_len <= d_res.bytes && total_len > copied) {
            ce = cudaMemcpyAsync((uint8_t*)d_res.p + copied, residues + copied, (size_t)(total_len - copied),
                                 cudaMemcpyHostToDevice, s);
            copied = total_len;
        }
    }
    static_assert((kMaxLen & (kMaxLen - 1)) == 0, "length check above");
    if (bad || too_short || ce != cudaSuccess) {
        cudaStreamSynchronize(s);  // the host arrays are borrowed for this call only
        if (ce != cudaSuccess) ctx->last_cuda = (int)ce, (void)cudaGetLastError();
        return bad ? TCRNET_ERR_LENGTH : too_short ? TCRNET_ERR_ARG : TCRNET_ERR_CUDA;
    }
    if (copied < total_len && (!d_res.p || d_res.bytes < (size_t)total_len)) {
        if (copied) cudaStreamSynchronize(s);  // (copies into the buffer that is replaced)
        copied = 0;
    }
    rc = dev_reserve(ctx, d_res, (size_t)total_len);
    int launches = 0;
    if (rc == TCRNET_OK && copied < total_len) {
        cudaError_t e = cudaMemcpyAsync((uint8_t*)d_res.p + copied, residues + copied, (size_t)(total_len - copied),
                                        cudaMemcpyHostToDevice, s);
        if (e != cudaSuccess) {
            ctx->last_cuda = (int)e;
            (void)cudaGetLastError();
            rc = TCRNET_ERR_CUDA;
        }
    }
    if (rc == TCRNET_OK)
        rc = load_from_device(ctx, (const uint8_t*)d_res.p, (const int32_t*)d_len.p, n, total_len, &launches);
    if (rc == TCRNET_OK) {
        cudaError_t e = cudaSuccess;
        ctx->stats.ms_load = 0.f;
        if (ctx->timing >= 2) {
            e = cudaEventRecord(ctx->ev[1], ctx->stream);
            if (e == cudaSuccess) e = cudaEventSynchronize(ctx->ev[1]);
            if (e == cudaSuccess) e = cudaEventElapsedTime(&ctx->stats.ms_load, ctx->ev[0], ctx->ev[1]);
        }
        if (e != cudaSuccess) {
            ctx->last_cuda = (int)e;
            (void)cudaGetLastError();
            rc = TCRNET_ERR_CUDA;
            drop_load(ctx);
        }
    }
    if (rc != TCRNET_OK) cudaStreamSynchronize(ctx->stream);  // the host arrays are borrowed for this call only
    ctx->stats.launches_load = launches;
    return rc;
}

int tcrnet_build(tcrnet_ctx* ctx, int l_max, int64_t* n_edges_out) {
    if (!ctx) return TCRNET_ERR_ARG;
    if (!ctx->loaded) return TCRNET_ERR_STATE;
    if (l_max < 0 || l_max > kMaxLen) return TCRNET_ERR_LMAX;
    TRY_CUDA(cudaSetDevice(ctx->device));
    drop_build(ctx);
    int launches = 0;
    TRY(distance_phase(ctx, l_max, 0, 1, &launches, /*assemble_too=*/true));
    if (ctx->assembled) TRY(assemble_finish(ctx, ctx->n_keys, (const unsigned long long*)ctx->keys_b.p, &launches));
    else TRY(assemble_phase(ctx, ctx->n_keys, true, &launches));
    tcrnet_stats& st = ctx->stats;
    st.ms_distance = st.ms_build = 0.f;
    if (ctx->timing >= 2) {
        TRY_CUDA(cudaEventElapsedTime(&st.ms_distance, ctx->ev[0], ctx->ev[1]));
        TRY_CUDA(cudaEventElapsedTime(&st.ms_build, ctx->ev[0], ctx->ev[3]));
    }
    st.launches_build = launches;
    ctx->built_l_max = l_max;
    if (n_edges_out) *n_edges_out = ctx->n_edges;
    return TCRNET_OK;
}

int tcrnet_build_shard(tcrnet_ctx* ctx, int l_max, int shard, int n_shards, const uint64_t** keys_dev,
                       int64_t* n_keys_out) {
    if (!ctx || n_shards < 1 || shard < 0 || shard >= n_shards) return TCRNET_ERR_ARG;
    if (!ctx->loaded) return TCRNET_ERR_STATE;
    if (l_max < 0 || l_max > kMaxLen) return TCRNET_ERR_LMAX;
    TRY_CUDA(cudaSetDevice(ctx->device));
    drop_build(ctx);
    int launches = 0;
    TRY(distance_phase(ctx, l_max, shard, n_shards, &launches));
    tcrnet_stats& st = ctx->stats;
    st.ms_distance = 0.f;
    if (ctx->timing >= 2) {
        TRY_CUDA(cudaEventSynchronize(ctx->ev[1]));
        TRY_CUDA(cudaEventElapsedTime(&st.ms_distance, ctx->ev[0], ctx->ev[1]));
    }
    st.ms_sort = st.ms_csr = 0.f;
    st.ms_build = st.ms_distance;
    st.launches_build = launches;
    st.n_edges = ctx->n_keys;
    ctx->have_keys = true;
    ctx->built_l_max = l_max;
    if (keys_dev) *keys_dev = ctx->n_keys ? (const uint64_t*)ctx->keys_a.p : nullptr;
    if (n_keys_out) *n_keys_out = ctx->n_keys;
    return TCRNET_OK;
}

int tcrnet_assemble(tcrnet_ctx* ctx, const uint64_t* keys_dev, int64_t n_keys, int64_t* n_edges_out) {
    if (!ctx || n_keys < 0 || (n_keys > 0 && !keys_dev)) return TCRNET_ERR_ARG;
    if (!ctx->loaded) return TCRNET_ERR_STATE;
    if (n_keys > ctx->edge_limit) return TCRNET_ERR_EDGE_OVERFLOW;
    TRY_CUDA(cudaSetDevice(ctx->device));
    cudaStream_t s = ctx->stream;
    const bool in_place = n_keys > 0 && keys_dev == (const uint64_t*)ctx->keys_a.p;
    if (in_place && !(ctx->have_keys && n_keys <= ctx->n_keys)) return TCRNET_ERR_ARG;
    ctx->built = false;
    ctx->have_dist = false;
    drop_observables(ctx);
    int launches = 0;
    if (!in_place) {
        // keys_dev may not alias the context's buffers: reserve first (contents are not preserved), then copy
        ctx->have_keys = false;
        TRY(dev_reserve(ctx, ctx->keys_a, sizeof(unsigned long long) * (size_t)std::max<int64_t>(n_keys, 1)));
        if (n_keys)
            TRY_CUDA(cudaMemcpyAsync(ctx->keys_a.p, keys_dev, sizeof(unsigned long long) * (size_t)n_keys,
                                     cudaMemcpyDeviceToDevice, s));
    }
    HostCtrl* dc = d_ctrl(ctx);
    TRY_CUDA(cudaMemsetAsync(&dc->flags, 0, sizeof(uint32_t), s));
    TRY_CUDA(launch_validate_keys((const unsigned long long*)ctx->keys_a.p, n_keys, ctx->n, &dc->flags, s, &launches));
    TRY_CUDA(cudaMemcpyAsync(&ctx->h_ctrl->flags, &dc->flags, sizeof(uint32_t), cudaMemcpyDeviceToHost, s));
    TRY_CUDA(rec(ctx, 1, 2));
    TRY_CUDA(cudaStreamSynchronize(s));
    if (ctx->h_ctrl->flags) return TCRNET_ERR_ARG;
    TRY(assemble_phase(ctx, n_keys, false, &launches));
    ctx->stats.launches_build = launches;
    ctx->stats.ms_build = 0.f;
    if (ctx->timing >= 2) TRY_CUDA(cudaEventElapsedTime(&ctx->stats.ms_build, ctx->ev[1], ctx->ev[3]));
    if (n_edges_out) *n_edges_out = ctx->n_edges;
    return TCRNET_OK;
}

int tcrnet_edge_distances(tcrnet_ctx* ctx, const uint8_t** dist_dev) {
    if (!ctx || !dist_dev) return TCRNET_ERR_ARG;
    if (!ctx->built) return TCRNET_ERR_STATE;
    TRY_CUDA(cudaSetDevice(ctx->device));
    int launches = 0;
    TRY(ensure_edge_distances(ctx, &launches));
    TRY_CUDA(cudaStreamSynchronize(ctx->stream));
    *dist_dev = ctx->n_edges ? (const uint8_t*)ctx->edge_dist.p : nullptr;
    return TCRNET_OK;
}

int tcrnet_restrict(tcrnet_ctx* ctx, int l_max, int64_t* n_edges_out) {
    if (!ctx) return TCRNET_ERR_ARG;
    if (!ctx->built) return TCRNET_ERR_STATE;
    if (l_max < 0 || l_max > ctx->built_l_max) return TCRNET_ERR_LMAX;
    TRY_CUDA(cudaSetDevice(ctx->device));
    cudaStream_t s = ctx->stream;
    int launches = 0;
    TRY(ensure_edge_distances(ctx, &launches));
    const int64_t e_old = ctx->n_edges;
    int64_t e_new = 0;
    drop_observables(ctx);
    TRY_CUDA(cudaEventRecord(ctx->ev[1], s));
    if (e_old > 0) {
        TRY(dev_reserve(ctx, ctx->flags, sizeof(uint32_t) * (size_t)e_old));
        TRY(dev_reserve(ctx, ctx->flag_pos, sizeof(uint32_t) * (size_t)(e_old + 1)));
        TRY(dev_reserve(ctx, ctx->scan_scratch, scan_scratch_bytes(e_old)));
        TRY(dev_reserve(ctx, ctx->keys_a, sizeof(unsigned long long) * (size_t)e_old));
        TRY(dev_reserve(ctx, ctx->edge_dist_b, (size_t)e_old));
        TRY_CUDA(launch_restrict_flags((const uint8_t*)ctx->edge_dist.p, e_old, l_max, (uint32_t*)ctx->flags.p, s, &launches));
        TRY_CUDA(exclusive_scan_u32_total((const uint32_t*)ctx->flags.p, (uint32_t*)ctx->flag_pos.p, e_old,
                                          ctx->scan_scratch.p, s, &launches));
        // (edge_row belongs to the CSR being restricted: ensure_edge_distances wrote it, or the restriction before)
        TRY_CUDA(launch_restrict_compact((const int32_t*)ctx->edge_row.p, (const int32_t*)ctx->col.p,
                                         (const uint8_t*)ctx->edge_dist.p, e_old, (const uint32_t*)ctx->flags.p,
                                         (const uint32_t*)ctx->flag_pos.p, (unsigned long long*)ctx->keys_a.p,
                                         (uint8_t*)ctx->edge_dist_b.p, s, &launches));
        uint32_t total = 0;
        TRY_CUDA(cudaMemcpyAsync(&ctx->h_ctrl->flags, (const uint32_t*)ctx->flag_pos.p + e_old, sizeof(uint32_t),
                                 cudaMemcpyDeviceToHost, s));
        TRY_CUDA(cudaStreamSynchronize(s));
        total = ctx->h_ctrl->flags;
        e_new = (int64_t)total;
        std::swap(ctx->edge_dist, ctx->edge_dist_b);
    }
    // the compaction is stable, so the keys are already sorted: CSR + degrees directly
    TRY_CUDA(cudaEventRecord(ctx->ev[2], s));
    TRY_CUDA(launch_csr((const unsigned long long*)ctx->keys_a.p, e_new, ctx->n, (int64_t*)ctx->row_ptr.p,
                        (int32_t*)ctx->col.p, (int32_t*)ctx->deg.p, s, &launches));
    // the labels stay valid for the restricted CSR (compacted above); so must the first indices of its edges
    if (e_new > 0) TRY_CUDA(launch_edge_rows((const int64_t*)ctx->row_ptr.p, ctx->n, (int32_t*)ctx->edge_row.p, s, &launches));
    TRY_CUDA(cudaEventRecord(ctx->ev[3], s));
    TRY_CUDA(cudaEventSynchronize(ctx->ev[3]));
    tcrnet_stats& st = ctx->stats;
    st.ms_distance = 0.f;
    TRY_CUDA(cudaEventElapsedTime(&st.ms_sort, ctx->ev[1], ctx->ev[2]));
    TRY_CUDA(cudaEventElapsedTime(&st.ms_csr, ctx->ev[2], ctx->ev[3]));
    TRY_CUDA(cudaEventElapsedTime(&st.ms_build, ctx->ev[1], ctx->ev[3]));
    st.launches_build = launches;
    st.l_max = l_max;
    st.n_edges = e_new;
    ctx->n_edges = e_new;
    ctx->built_l_max = l_max;
    ctx->have_keys = false;
    if (n_edges_out) *n_edges_out = e_new;
    return TCRNET_OK;
}

int tcrnet_csr(tcrnet_ctx* ctx, const int64_t** row_ptr_dev, const int32_t** col_dev) {
    if (!ctx) return TCRNET_ERR_ARG;
    if (!ctx->built) return TCRNET_ERR_STATE;
    if (row_ptr_dev) *row_ptr_dev = (const int64_t*)ctx->row_ptr.p;
    if (col_dev) *col_dev = ctx->n_edges ? (const int32_t*)ctx->col.p : nullptr;
    return TCRNET_OK;
}

int tcrnet_degrees(tcrnet_ctx* ctx, const int32_t** deg_dev) {
    if (!ctx || !deg_dev) return TCRNET_ERR_ARG;
    if (!ctx->built) return TCRNET_ERR_STATE;
    *deg_dev = (const int32_t*)ctx->deg.p;
    return TCRNET_OK;
}

int tcrnet_copy_csr(tcrnet_ctx* ctx, int64_t* row_ptr_host, int32_t* col_host, int32_t* deg_host) {
    if (!ctx) return TCRNET_ERR_ARG;
    if (!ctx->built) return TCRNET_ERR_STATE;
    TRY_CUDA(cudaSetDevice(ctx->device));
    cudaStream_t s = ctx->stream;
    if (row_ptr_host)
        TRY_CUDA(cudaMemcpyAsync(row_ptr_host, ctx->row_ptr.p, sizeof(int64_t) * (size_t)(ctx->n + 1), cudaMemcpyDeviceToHost, s));
    if (col_host && ctx->n_edges)
        TRY_CUDA(cudaMemcpyAsync(col_host, ctx->col.p, sizeof(int32_t) * (size_t)ctx->n_edges, cudaMemcpyDeviceToHost, s));
    if (deg_host)
        TRY_CUDA(cudaMemcpyAsync(deg_host, ctx->deg.p, sizeof(int32_t) * (size_t)ctx->n, cudaMemcpyDeviceToHost, s));
    TRY_CUDA(cudaStreamSynchronize(s));
    return TCRNET_OK;
}

int tcrnet_set_option(tcrnet_ctx* ctx, int option, int64_t value) {
    if (!ctx) return TCRNET_ERR_ARG;
    switch (option) {
        case TCRNET_OPT_EARLY_EXIT:
            if (value != 0 && value != 1) return TCRNET_ERR_ARG;
            ctx->early_exit = (int)value;
            return TCRNET_OK;
        case TCRNET_OPT_FIRST_CHECK:
            if (value != 0 && (value < 3 || value > 8)) return TCRNET_ERR_ARG;
            ctx->first_check_opt = (int)value;
            return TCRNET_OK;
        case TCRNET_OPT_EDGE_CAPACITY:
            if (value < 0) return TCRNET_ERR_ARG;
            ctx->edge_capacity_opt = value;
            if (value > 0) dev_free(ctx, ctx->keys_a);  // honour a smaller capacity next time
            return TCRNET_OK;
        case TCRNET_OPT_EDGE_LIMIT:
            if (value < 1 || value > ((int64_t)1 << 31)) return TCRNET_ERR_ARG;
            ctx->edge_limit = value;
            return TCRNET_OK;
        case TCRNET_OPT_COUNT_WORK:
            if (value != 0 && value != 1) return TCRNET_ERR_ARG;
            ctx->count_work = (int)value;
            return TCRNET_OK;
        case TCRNET_OPT_TEXT_CHUNK:
            if (value < kTQ || value % kTQ != 0 || value > (1 << 20)) return TCRNET_ERR_ARG;
            ctx->tchunk = (int)value;
            return TCRNET_OK;
        case TCRNET_OPT_PREFIX_TRIE:
            if (value != 0 && value != 1) return TCRNET_ERR_ARG;
            ctx->prefix_trie = (int)value;
            return TCRNET_OK;
        case TCRNET_OPT_N_QUERY:
            if (value < 0 || value > 0x7ffffffeLL) return TCRNET_ERR_ARG;
            ctx->n_query = value;
            return TCRNET_OK;
        case TCRNET_OPT_DEDUP:
            if (value != 0 && value != 1) return TCRNET_ERR_ARG;
            ctx->dedup = (int)value;
            ctx->dedup_pause = 0;
            return TCRNET_OK;
        case TCRNET_OPT_SEGMENT_JOIN:
            if (value < -1 || value > 1) return TCRNET_ERR_ARG;
            ctx->segment_join = (int)value;
            return TCRNET_OK;
        case TCRNET_OPT_FAST_L1:
            if (value != 0 && value != 1) return TCRNET_ERR_ARG;
            ctx->fast_l1 = (int)value;
            return TCRNET_OK;
        case TCRNET_OPT_TIMING:
            if (value < 0 || value > 2) return TCRNET_ERR_ARG;
            ctx->timing = (int)value;
            return TCRNET_OK;
        case TCRNET_OPT_TRIE_CHUNK:
            if (value < kTQ || value % kTQ != 0 || value > (1 << 24)) return TCRNET_ERR_ARG;
            ctx->trie_chunk = (int)value;
            return TCRNET_OK;
        default: return TCRNET_ERR_ARG;
    }
}

int tcrnet_get_stats(tcrnet_ctx* ctx, tcrnet_stats* out) {
    if (!ctx || !out) return TCRNET_ERR_ARG;
    *out = ctx->stats;
    return TCRNET_OK;
}

int tcrnet_probe_int32(tcrnet_ctx* ctx, int kind, double* ops_per_s, double* sm_clock_mhz) {
    if (!ctx || kind < 0 || kind > 5 || !ops_per_s) return TCRNET_ERR_ARG;
    TRY_CUDA(cudaSetDevice(ctx->device));
    HostCtrl* dc = d_ctrl(ctx);
    float ms = 0.f;
    TRY_CUDA(launch_probe(kind, ctx->n_sm, dc->probe, &ms, ctx->stream));
    TRY_CUDA(cudaMemcpyAsync(ctx->h_ctrl->probe, dc->probe, sizeof(unsigned long long) * 3, cudaMemcpyDeviceToHost, ctx->stream));
    TRY_CUDA(cudaStreamSynchronize(ctx->stream));
    *ops_per_s = (double)ctx->h_ctrl->probe[0] / ((double)ms * 1e-3);
    if (sm_clock_mhz) *sm_clock_mhz = (double)ctx->h_ctrl->probe[1] / ((double)ms * 1e3);
    return TCRNET_OK;
}

int tcrnet_last_cuda_error(tcrnet_ctx* ctx) { return ctx ? ctx->last_cuda : 0; }

}  // extern "C"

// C ABI of libtcrnet_b200.so (include/tcrnet.h): context, memory, the host half of the tile
// scheduler (step A2) and the orchestration of steps A1-A6 on one CUDA stream.
#include <algorithm>
#include <cstddef>
#include <cstring>
#include <new>
#include <vector>

#include "tcrnet_internal.h"

using namespace tcrnet;

namespace {

struct DevBuf {
    void* p = nullptr;
    size_t bytes = 0;
};

struct HostCtrl {  // pinned mirror of the small device control block
    unsigned long long hist[kNumLen];
    unsigned long long edge_count;
    unsigned long long work[4];
    unsigned long long probe[3];
    uint32_t flags;
    uint32_t pad_;
    uint32_t trie_counts[8];          // [k] = nodes of trie level k
    uint32_t trie_root[kNumLen + 1];  // [L] = first level-1 node of length bucket L (non-empty buckets)
};

}  // namespace

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
    int trie_chunk = 32768;

    // load state
    bool loaded = false;
    int64_t n = 0, total_len = 0;
    int64_t hist[kNumLen] = {};
    LengthTable lt{};
    int pat_stride = 0;
    DevBuf perm, pat, txt, trie;
    TrieLevels trie_levels{};
    uint32_t trie_root[kNumLen + 1] = {};  // level-1 node range of bucket L: [trie_root[L], trie_root[L+1])

    // build state
    bool built = false;
    int64_t n_edges = 0;
    DevBuf keys_a, keys_b, split_hist, split_hist_scanned, scan_scratch, rows, row_ptr, col, deg;

    DevBuf ctrl;               // device HostCtrl
    HostCtrl* h_ctrl = nullptr;  // pinned
    cudaEvent_t ev[6] = {};
    tcrnet_stats stats{};
};

namespace {

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

HostCtrl* d_ctrl(tcrnet_ctx* ctx) { return static_cast<HostCtrl*>(ctx->ctrl.p); }

int bits_for(int64_t max_value) {  // number of bits needed to represent max_value (>= 1)
    int b = 1;
    while (b < 63 && (max_value >> b) != 0) ++b;
    return b;
}

void drop_build(tcrnet_ctx* ctx) {
    ctx->built = false;
    ctx->n_edges = 0;
}

void drop_load(tcrnet_ctx* ctx) {
    drop_build(ctx);
    ctx->loaded = false;
    ctx->n = 0;
}

// Steps A1: everything after the raw arrays are in device memory.
int load_from_device(tcrnet_ctx* ctx, const uint8_t* d_res, const int32_t* d_len, int64_t n, int64_t total_len,
                     int* launches) {
    cudaStream_t s = ctx->stream;
    HostCtrl* dc = d_ctrl(ctx);
    TRY_CUDA(cudaMemsetAsync(dc, 0, sizeof(HostCtrl), s));
    TRY_CUDA(launch_length_hist(d_len, n, dc->hist, &dc->flags, s, launches));
    TRY_CUDA(cudaMemcpyAsync(ctx->h_ctrl, dc, sizeof(HostCtrl), cudaMemcpyDeviceToHost, s));
    TRY_CUDA(cudaStreamSynchronize(s));
    if (ctx->h_ctrl->flags & kFlagBadLength) return TCRNET_ERR_LENGTH;
    int64_t sum = 0, cnt = 0;
    int min_len = kMaxLen, max_len = 0;
    for (int l = 0; l < kNumLen; ++l) {
        ctx->hist[l] = (int64_t)ctx->h_ctrl->hist[l];
        if (ctx->hist[l]) {
            min_len = std::min(min_len, l);
            max_len = std::max(max_len, l);
        }
        sum += ctx->hist[l] * l;
        cnt += ctx->hist[l];
    }
    if (cnt != n || sum != total_len) return TCRNET_ERR_ARG;

    // per-length layout
    LengthTable& lt = ctx->lt;
    int64_t pos = 0, words = 0;
    for (int l = 0; l < kNumLen; ++l) {
        lt.start[l] = (int32_t)pos;
        lt.txt_base[l] = words;
        lt.row_words[l] = (l + 3) & ~3;
        pos += ctx->hist[l];
        words += ctx->hist[l] * lt.row_words[l];
    }
    lt.start[kNumLen] = (int32_t)pos;
    lt.txt_base[kNumLen] = words;
    ctx->pat_stride = (max_len + 15) & ~15;

    // offsets, stable sort by (length, row), re-layout
    DevBuf offsets;
    const int64_t blocks = split_num_blocks(n);
    int rc = dev_reserve(ctx, offsets, sizeof(int64_t) * (size_t)(n + 1));
    if (rc == TCRNET_OK) rc = dev_reserve(ctx, ctx->scan_scratch, std::max(scan_scratch_bytes(n), scan_scratch_bytes(256 * blocks)));
    if (rc == TCRNET_OK) rc = dev_reserve(ctx, ctx->split_hist, sizeof(uint32_t) * 256 * (size_t)blocks);
    if (rc == TCRNET_OK) rc = dev_reserve(ctx, ctx->split_hist_scanned, sizeof(uint32_t) * 256 * (size_t)blocks);
    if (rc == TCRNET_OK) rc = dev_reserve(ctx, ctx->perm, sizeof(int32_t) * (size_t)n);
    if (rc == TCRNET_OK) rc = dev_reserve(ctx, ctx->pat, (size_t)n * ctx->pat_stride);
    if (rc == TCRNET_OK) rc = dev_reserve(ctx, ctx->txt, sizeof(uint32_t) * (size_t)(words + 4));
    if (rc != TCRNET_OK) {
        dev_free(ctx, offsets);
        return rc;
    }
    // Sort key: (length, first kSortPrefix residues, row).  LSD: least significant digit first, every
    // pass stable.  The sub-order inside a length bucket is free (results are mapped back through
    // perm); the lexicographic one makes the 32 patterns of a warp share their first residues, so the
    // early-exit test of the distance kernel fails or holds for the whole warp at once.
    DevBuf perm_tmp;
    rc = dev_reserve(ctx, perm_tmp, sizeof(int32_t) * (size_t)n);
    if (rc != TCRNET_OK) {
        dev_free(ctx, offsets);
        return rc;
    }
    cudaError_t e = exclusive_scan_i32_to_i64(d_len, (int64_t*)offsets.p, n, true, ctx->scan_scratch.p, s, launches);
    {
        // kSortPrefix + 1 passes ping-pong between the two buffers; arrange for the last to land in ctx->perm
        int32_t* bufs[2] = {(int32_t*)ctx->perm.p, (int32_t*)perm_tmp.p};
        int cur = kSortPrefix & 1;  // buffer written by the first pass
        const int32_t* in = nullptr;
        for (int k = kSortPrefix - 1; k >= 0 && e == cudaSuccess; --k) {
            e = split_by_residue(d_res, (const int64_t*)offsets.p, d_len, in, k, n, bufs[cur],
                                 (uint32_t*)ctx->split_hist.p, (uint32_t*)ctx->split_hist_scanned.p,
                                 ctx->scan_scratch.p, s, launches);
            in = bufs[cur];
            cur ^= 1;
        }
        if (e == cudaSuccess)
            e = split_by_length(d_len, in, n, bufs[cur], (uint32_t*)ctx->split_hist.p,
                                (uint32_t*)ctx->split_hist_scanned.p, ctx->scan_scratch.p, s, launches);
        // cur is now the index of the buffer holding the final order
        if (bufs[cur] != (int32_t*)ctx->perm.p) e = e == cudaSuccess ? cudaErrorUnknown : e;
    }
    if (e == cudaSuccess)
        e = launch_pack(d_res, (const int64_t*)offsets.p, d_len, (const int32_t*)ctx->perm.p, n, lt, ctx->pat_stride,
                        (uint8_t*)ctx->pat.p, (uint32_t*)ctx->txt.p, &dc->flags, s, launches);
    // prefix trie over the sorted texts (trie.cu); scratch: lcp8 + per-tile counts
    DevBuf trie_scratch;
    if (e == cudaSuccess) {
        size_t node_total = 0, level_off[kTrieDepth + 1] = {};
        for (int k = 1; k <= kTrieDepth; ++k) {
            level_off[k] = node_total;
            node_total += (size_t)trie_level_capacity(n, k);
        }
        const size_t lcp_bytes = (((size_t)n + 15) & ~(size_t)15) + 256;  // keeps the tile counts aligned
        rc = dev_reserve(ctx, ctx->trie, node_total * sizeof(TrieNode));
        if (rc == TCRNET_OK) rc = dev_reserve(ctx, trie_scratch, lcp_bytes + (size_t)trie_tiles(n) * 8 * sizeof(uint32_t));
        if (rc == TCRNET_OK) {
            for (int k = 1; k <= kTrieDepth; ++k) ctx->trie_levels.p[k] = (TrieNode*)ctx->trie.p + level_off[k];
            ctx->trie_levels.p[0] = nullptr;
            e = launch_trie_build((const uint32_t*)ctx->txt.p, lt, n, (uint8_t*)trie_scratch.p,
                                  (uint32_t*)((uint8_t*)trie_scratch.p + (lcp_bytes & ~(size_t)255)), ctx->trie_levels,
                                  dc->trie_counts, dc->trie_root, s, launches);
        }
    }
    if (rc == TCRNET_OK && e == cudaSuccess)
        e = cudaMemcpyAsync(&ctx->h_ctrl->flags, &dc->flags,
                            sizeof(HostCtrl) - offsetof(HostCtrl, flags), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    dev_free(ctx, offsets);
    dev_free(ctx, perm_tmp);
    dev_free(ctx, trie_scratch);
    if (rc != TCRNET_OK) return rc;
    TRY_CUDA(e);
    if (ctx->h_ctrl->flags & kFlagBadResidue) return TCRNET_ERR_RESIDUE;
    // level-1 node range of every bucket (empty buckets get an empty range)
    ctx->trie_root[kNumLen] = ctx->h_ctrl->trie_counts[1];
    for (int l = kNumLen - 1; l >= 0; --l)
        ctx->trie_root[l] = ctx->hist[l] ? ctx->h_ctrl->trie_root[l] : ctx->trie_root[l + 1];
    ctx->stats.trie_nodes = 0;
    for (int k = 1; k <= kTrieDepth; ++k) ctx->stats.trie_nodes += ctx->h_ctrl->trie_counts[k];

    ctx->n = n;
    ctx->total_len = total_len;
    ctx->stats.n = n;
    ctx->stats.total_len = total_len;
    ctx->stats.min_len = min_len;
    ctx->stats.max_len = max_len;
    ctx->loaded = true;
    return TCRNET_OK;
}

// The four launches of the distance step: {chunk kernel, trie kernel} x {32-bit, 64-bit words}.
struct Schedule {
    struct Part {
        std::vector<WorkRow> rows;
        int64_t items = 0;
        int max_rw = 4;
    };
    Part part[2][2];  // [trie][wide]
    int first_test = 0;  // trie kernel: first level with an early-exit test (0: trie not used)
};

// Step A2, host side: the (pattern bucket, text bucket) pairs with len_t - len_p in 0..l_max.
void make_schedule(const tcrnet_ctx* ctx, int l_max, int first_check, Schedule& sch, tcrnet_stats& st) {
    const LengthTable& lt = ctx->lt;
    st.pairs_kept = st.cells_kept = st.columns_kept = st.cells_all = 0;
    long double cells_all = 0;
    {
        long double sum_len = 0, sum_sq = 0;  // sum over unordered pairs of la*lb = ((sum l)^2 - sum l^2) / 2
        for (int l = 1; l < kNumLen; ++l) {
            sum_len += (long double)ctx->hist[l] * l;
            sum_sq += (long double)ctx->hist[l] * l * l;
        }
        cells_all = (sum_len * sum_len - sum_sq) / 2;
    }
    st.cells_all = (int64_t)cells_all;
    st.pairs_all = ctx->n * (ctx->n - 1) / 2;
    // The trie kernel serves the rows whose early exit can act inside the trie: first test level
    // <= kTrieDepth and at least one text column beyond the trie.
    const bool use_trie = ctx->prefix_trie && first_check >= 3 && first_check <= kTrieDepth;
    sch.first_test = use_trie ? first_check : 0;
    for (int m = 1; m < kNumLen; ++m) {
        if (!ctx->hist[m]) continue;
        for (int n = m; n <= std::min(kMaxLen, m + l_max); ++n) {
            if (!ctx->hist[n]) continue;
            const int64_t pc = ctx->hist[m], tc = ctx->hist[n];
            const int64_t pairs = (m == n) ? pc * (pc - 1) / 2 : pc * tc;
            st.pairs_kept += pairs;
            st.cells_kept += pairs * m * n;
            st.columns_kept += pairs * n;
            if (pairs == 0) continue;
            const bool trie = use_trie && n > kTrieDepth;
            WorkRow r{};
            r.txt_base = lt.txt_base[n];
            r.p_start = lt.start[m];
            r.p_count = (int32_t)pc;
            r.t_start = lt.start[n];
            r.t_count = (int32_t)tc;
            r.m = m;
            r.n = n;
            r.row_words = lt.row_words[n];
            r.tchunk = trie ? ctx->trie_chunk : ctx->tchunk;
            r.n_tchunks = (int32_t)((tc + r.tchunk - 1) / r.tchunk);
            r.diag = (m == n) ? 1 : 0;
            r.root_begin = ctx->trie_root[n];
            r.root_end = ctx->trie_root[n + 1];
            sch.part[trie ? 1 : 0][m <= 32 ? 0 : 1].rows.push_back(r);
        }
    }
    for (auto& by_kernel : sch.part)
        for (Schedule::Part& part : by_kernel) {
            auto n_items = [](const WorkRow& r) { return (int64_t)((r.p_count + kTQ - 1) / kTQ) * r.n_tchunks; };
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
}

int run_distance(tcrnet_ctx* ctx, const Schedule& sch, int l_max, int first_check, uint64_t cap, int* launches) {
    cudaStream_t s = ctx->stream;
    HostCtrl* dc = d_ctrl(ctx);
    TRY_CUDA(cudaMemsetAsync(&dc->edge_count, 0, sizeof(unsigned long long) * 5, s));  // edge_count + work[4]
    DistanceParams p{};
    p.l_max = l_max;
    p.pat_stride = ctx->pat_stride;
    p.txt = (const uint32_t*)ctx->txt.p;
    p.pat = (const uint8_t*)ctx->pat.p;
    p.perm = (const int32_t*)ctx->perm.p;
    p.edges = (unsigned long long*)ctx->keys_a.p;
    p.edge_count = &dc->edge_count;
    p.edge_cap = cap;
    p.work = dc->work;
    for (int k = 0; k <= kTrieDepth; ++k) p.trie[k] = ctx->trie_levels.p[k];
    const WorkRow* d_rows = (const WorkRow*)ctx->rows.p;
    for (int trie = 1; trie >= 0; --trie)
        for (int wide = 0; wide < 2; ++wide) {
            const Schedule::Part& part = sch.part[trie][wide];
            if (!part.rows.empty()) {
                p.rows = d_rows;
                p.n_rows = (int32_t)part.rows.size();
                if (trie)
                    TRY_CUDA(launch_distance_trie(p, part.items, wide != 0, ctx->count_work != 0, s, launches));
                else
                    TRY_CUDA(launch_distance(p, part.items, wide != 0, first_check, ctx->count_work != 0, part.max_rw, s, launches));
            }
            d_rows += part.rows.size();
        }
    TRY_CUDA(cudaMemcpyAsync(&ctx->h_ctrl->edge_count, &dc->edge_count, sizeof(unsigned long long) * 5,
                             cudaMemcpyDeviceToHost, s));
    TRY_CUDA(cudaStreamSynchronize(s));
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
    for (int i = 0; e == cudaSuccess && i < 6; ++i) e = cudaEventCreate(&ctx->ev[i]);
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
    DevBuf* bufs[] = {&ctx->perm, &ctx->pat, &ctx->txt, &ctx->trie, &ctx->keys_a, &ctx->keys_b, &ctx->split_hist,
                      &ctx->split_hist_scanned, &ctx->scan_scratch, &ctx->rows, &ctx->row_ptr, &ctx->col,
                      &ctx->deg, &ctx->ctrl};
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
    drop_load(ctx);
    int launches = 0;
    TRY_CUDA(cudaEventRecord(ctx->ev[0], ctx->stream));
    TRY(load_from_device(ctx, residues_dev, lengths_dev, n, total_len, &launches));
    TRY_CUDA(cudaEventRecord(ctx->ev[1], ctx->stream));
    TRY_CUDA(cudaEventSynchronize(ctx->ev[1]));
    TRY_CUDA(cudaEventElapsedTime(&ctx->stats.ms_load, ctx->ev[0], ctx->ev[1]));
    ctx->stats.launches_load = launches;
    return TCRNET_OK;
}

int tcrnet_load(tcrnet_ctx* ctx, const uint8_t* residues, const int32_t* lengths, int64_t n) {
    if (!ctx || !residues || !lengths || n < 1 || n > 0x7ffffffeLL) return TCRNET_ERR_ARG;
    TRY_CUDA(cudaSetDevice(ctx->device));
    drop_load(ctx);
    // the host pass only sizes the copy; validation proper happens on the device
    int64_t total_len = 0;
    for (int64_t i = 0; i < n; ++i) {
        if (lengths[i] < 1 || lengths[i] > kMaxLen) return TCRNET_ERR_LENGTH;
        total_len += lengths[i];
    }
    DevBuf d_res, d_len;
    int rc = dev_reserve(ctx, d_res, (size_t)total_len);
    if (rc == TCRNET_OK) rc = dev_reserve(ctx, d_len, sizeof(int32_t) * (size_t)n);
    int launches = 0;
    if (rc == TCRNET_OK) {
        cudaStream_t s = ctx->stream;
        cudaError_t e = cudaEventRecord(ctx->ev[0], s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_res.p, residues, (size_t)total_len, cudaMemcpyHostToDevice, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_len.p, lengths, sizeof(int32_t) * (size_t)n, cudaMemcpyHostToDevice, s);
        if (e != cudaSuccess) {
            ctx->last_cuda = (int)e;
            (void)cudaGetLastError();
            rc = TCRNET_ERR_CUDA;
        }
    }
    if (rc == TCRNET_OK)
        rc = load_from_device(ctx, (const uint8_t*)d_res.p, (const int32_t*)d_len.p, n, total_len, &launches);
    if (rc == TCRNET_OK) {
        cudaError_t e = cudaEventRecord(ctx->ev[1], ctx->stream);
        if (e == cudaSuccess) e = cudaEventSynchronize(ctx->ev[1]);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ctx->stats.ms_load, ctx->ev[0], ctx->ev[1]);
        if (e != cudaSuccess) {
            ctx->last_cuda = (int)e;
            (void)cudaGetLastError();
            rc = TCRNET_ERR_CUDA;
            drop_load(ctx);
        }
    }
    cudaStreamSynchronize(ctx->stream);
    dev_free(ctx, d_res);
    dev_free(ctx, d_len);
    ctx->stats.launches_load = launches;
    return rc;
}

int tcrnet_build(tcrnet_ctx* ctx, int l_max, int64_t* n_edges_out) {
    if (!ctx) return TCRNET_ERR_ARG;
    if (!ctx->loaded) return TCRNET_ERR_STATE;
    if (l_max < 0 || l_max > kMaxLen) return TCRNET_ERR_LMAX;
    TRY_CUDA(cudaSetDevice(ctx->device));
    drop_build(ctx);
    cudaStream_t s = ctx->stream;
    tcrnet_stats& st = ctx->stats;
    int launches = 0;
    const int64_t n = ctx->n;

    // ---- A2: schedule ----
    int first_check = 0;
    if (ctx->early_exit) {
        first_check = ctx->first_check_opt ? ctx->first_check_opt : l_max + 2;
        first_check = std::max(3, std::min(8, first_check));
    }
    st.first_check = first_check;
    Schedule sch;
    make_schedule(ctx, l_max, first_check, sch, st);
    st.l_max = l_max;
    st.work_items = st.work_items_trie = 0;
    size_t n_rows = 0;
    for (int trie = 0; trie < 2; ++trie)
        for (int wide = 0; wide < 2; ++wide) {
            st.work_items += sch.part[trie][wide].items;
            if (trie) st.work_items_trie += sch.part[trie][wide].items;
            n_rows += sch.part[trie][wide].rows.size();
        }
    TRY(dev_reserve(ctx, ctx->rows, sizeof(WorkRow) * std::max<size_t>(n_rows, 1)));
    TRY_CUDA(cudaEventRecord(ctx->ev[0], s));
    {
        // same order as run_distance walks them: trie parts first
        WorkRow* dst = (WorkRow*)ctx->rows.p;
        for (int trie = 1; trie >= 0; --trie)
            for (int wide = 0; wide < 2; ++wide) {
                const std::vector<WorkRow>& rows = sch.part[trie][wide].rows;
                if (!rows.empty())
                    TRY_CUDA(cudaMemcpyAsync(dst, rows.data(), sizeof(WorkRow) * rows.size(), cudaMemcpyHostToDevice, s));
                dst += rows.size();
            }
    }

    // ---- A3-A5: distances + emission (second pass only if the edge buffer was too small) ----
    int64_t cap = ctx->edge_capacity_opt > 0 ? ctx->edge_capacity_opt : std::max<int64_t>((int64_t)1 << 20, 16 * n);
    cap = std::min(cap, ctx->edge_limit);
    cap = std::max<int64_t>(cap, 1);
    if (ctx->keys_a.p && (int64_t)(ctx->keys_a.bytes / 8) > cap) cap = std::min<int64_t>(ctx->keys_a.bytes / 8, ctx->edge_limit);
    TRY(dev_reserve(ctx, ctx->keys_a, sizeof(unsigned long long) * (size_t)cap));
    st.distance_passes = 1;
    TRY(run_distance(ctx, sch, l_max, first_check, (uint64_t)cap, &launches));
    int64_t n_edges = (int64_t)ctx->h_ctrl->edge_count;
    if (n_edges > ctx->edge_limit) return TCRNET_ERR_EDGE_OVERFLOW;
    if (n_edges > cap) {
        cap = n_edges;
        TRY(dev_reserve(ctx, ctx->keys_a, sizeof(unsigned long long) * (size_t)cap));
        st.distance_passes = 2;
        TRY(run_distance(ctx, sch, l_max, first_check, (uint64_t)cap, &launches));
        if ((int64_t)ctx->h_ctrl->edge_count != n_edges) return TCRNET_ERR_CUDA;  // cannot happen: same input
    }
    st.lane_columns_exec = (int64_t)ctx->h_ctrl->work[0];
    st.lane_tests_exec = (int64_t)ctx->h_ctrl->work[1];
    st.lane_pairs_exec = (int64_t)ctx->h_ctrl->work[2];
    st.lane_prefix_tests_exec = (int64_t)ctx->h_ctrl->work[3];
    TRY_CUDA(cudaEventRecord(ctx->ev[1], s));

    // ---- A6a: LSD radix sort of the keys (u << 32) | v over the significant bits only ----
    const unsigned long long* sorted = (const unsigned long long*)ctx->keys_a.p;
    if (n_edges > 1) {
        const int64_t blocks = split_num_blocks(n_edges);
        TRY(dev_reserve(ctx, ctx->keys_b, sizeof(unsigned long long) * (size_t)n_edges));
        TRY(dev_reserve(ctx, ctx->split_hist, sizeof(uint32_t) * 256 * (size_t)blocks));
        TRY(dev_reserve(ctx, ctx->split_hist_scanned, sizeof(uint32_t) * 256 * (size_t)blocks));
        TRY(dev_reserve(ctx, ctx->scan_scratch, scan_scratch_bytes(256 * blocks)));
        const int id_bits = bits_for(n - 1 > 0 ? n - 1 : 1);
        unsigned long long* a = (unsigned long long*)ctx->keys_a.p;
        unsigned long long* b = (unsigned long long*)ctx->keys_b.p;
        for (int half = 0; half < 2; ++half)
            for (int sh = 0; sh < id_bits; sh += 8) {
                TRY_CUDA(split_keys_u64(a, b, n_edges, 32 * half + sh, (uint32_t*)ctx->split_hist.p,
                                        (uint32_t*)ctx->split_hist_scanned.p, ctx->scan_scratch.p, s, &launches));
                std::swap(a, b);
            }
        sorted = a;
    }
    TRY_CUDA(cudaEventRecord(ctx->ev[2], s));

    // ---- A6b: CSR + degrees ----
    TRY(dev_reserve(ctx, ctx->row_ptr, sizeof(int64_t) * (size_t)(n + 1)));
    TRY(dev_reserve(ctx, ctx->col, sizeof(int32_t) * (size_t)std::max<int64_t>(n_edges, 1)));
    TRY(dev_reserve(ctx, ctx->deg, sizeof(int32_t) * (size_t)n));
    TRY_CUDA(launch_csr(sorted, n_edges, n, (int64_t*)ctx->row_ptr.p, (int32_t*)ctx->col.p, (int32_t*)ctx->deg.p, s, &launches));
    TRY_CUDA(cudaEventRecord(ctx->ev[3], s));
    TRY_CUDA(cudaEventSynchronize(ctx->ev[3]));
    TRY_CUDA(cudaEventElapsedTime(&st.ms_distance, ctx->ev[0], ctx->ev[1]));
    TRY_CUDA(cudaEventElapsedTime(&st.ms_sort, ctx->ev[1], ctx->ev[2]));
    TRY_CUDA(cudaEventElapsedTime(&st.ms_csr, ctx->ev[2], ctx->ev[3]));
    TRY_CUDA(cudaEventElapsedTime(&st.ms_build, ctx->ev[0], ctx->ev[3]));
    st.launches_build = launches;
    st.n_edges = n_edges;
    ctx->n_edges = n_edges;
    ctx->built = true;
    if (n_edges_out) *n_edges_out = n_edges;
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

// C ABI, network observables on the current CSR (include/tcrnet.h):
// tcrnet_degree_histogram, tcrnet_neighbor_degree, tcrnet_components, tcrnet_percolation.
// Host orchestration only; the kernels are in observables.cu.
#include <algorithm>
#include <vector>

#include "tcrnet_ctx.h"

namespace {

struct ObsCtrl {  // small device control block of the observables
    int32_t max_degree;
    uint32_t flag;
    unsigned long long lcc;
    unsigned long long n_comp;
};

ObsCtrl* d_obs(tcrnet_ctx* ctx) { return static_cast<ObsCtrl*>(ctx->obs_ctrl.p); }

int fetch_ctrl(tcrnet_ctx* ctx, ObsCtrl* host) {
    TRY_CUDA(cudaMemcpyAsync(host, ctx->obs_ctrl.p, sizeof(ObsCtrl), cudaMemcpyDeviceToHost, ctx->stream));
    TRY_CUDA(cudaStreamSynchronize(ctx->stream));
    return TCRNET_OK;
}

// hist[d], d = 0..max_degree, of the full network
int ensure_degree_hist(tcrnet_ctx* ctx, int* launches) {
    if (ctx->have_hist) return TCRNET_OK;
    cudaStream_t s = ctx->stream;
    TRY(dev_reserve(ctx, ctx->obs_ctrl, sizeof(ObsCtrl)));
    TRY_CUDA(cudaMemsetAsync(ctx->obs_ctrl.p, 0, sizeof(ObsCtrl), s));
    TRY_CUDA(launch_max_degree((const int32_t*)ctx->deg.p, ctx->n, &d_obs(ctx)->max_degree, s, launches));
    ObsCtrl h{};
    TRY(fetch_ctrl(ctx, &h));
    ctx->max_degree = h.max_degree;
    const size_t bytes = sizeof(unsigned long long) * ((size_t)h.max_degree + 1);
    TRY(dev_reserve(ctx, ctx->deg_hist, bytes));
    TRY_CUDA(cudaMemsetAsync(ctx->deg_hist.p, 0, bytes, s));
    TRY_CUDA(launch_degree_hist((const int32_t*)ctx->deg.p, ctx->n, nullptr, 0, (unsigned long long*)ctx->deg_hist.p, s,
                                launches));
    ctx->have_hist = true;
    return TCRNET_OK;
}

int ensure_components(tcrnet_ctx* ctx, int* launches) {
    if (ctx->have_cc) return TCRNET_OK;
    cudaStream_t s = ctx->stream;
    const int64_t n = ctx->n;
    TRY(dev_reserve(ctx, ctx->obs_ctrl, sizeof(ObsCtrl)));
    TRY(dev_reserve(ctx, ctx->cc_parent, sizeof(int32_t) * (size_t)n));
    TRY(dev_reserve(ctx, ctx->cc_count, sizeof(int32_t) * (size_t)n));
    TRY(dev_reserve(ctx, ctx->cc_label, sizeof(int32_t) * (size_t)n));
    TRY(dev_reserve(ctx, ctx->cc_size, sizeof(int32_t) * (size_t)n));
    TRY_CUDA(cudaMemsetAsync(&d_obs(ctx)->lcc, 0, 2 * sizeof(unsigned long long), s));
    TRY_CUDA(launch_components((const int64_t*)ctx->row_ptr.p, (const int32_t*)ctx->col.p, n, nullptr, 0,
                               (int32_t*)ctx->cc_parent.p, (int32_t*)ctx->cc_count.p, (int32_t*)ctx->cc_label.p, nullptr,
                               &d_obs(ctx)->lcc, &d_obs(ctx)->n_comp, s, launches));
    TRY_CUDA(launch_component_sizes(n, (const int32_t*)ctx->cc_label.p, (const int32_t*)ctx->cc_count.p,
                                    (int32_t*)ctx->cc_size.p, s, launches));
    ObsCtrl h{};
    TRY(fetch_ctrl(ctx, &h));
    ctx->lcc = (int64_t)h.lcc;
    ctx->n_components = (int64_t)h.n_comp;
    ctx->have_cc = true;
    return TCRNET_OK;
}

}  // namespace

extern "C" {

int tcrnet_degree_histogram(tcrnet_ctx* ctx, const int64_t** hist_dev, int32_t* max_degree_out) {
    if (!ctx) return TCRNET_ERR_ARG;
    if (!ctx->built) return TCRNET_ERR_STATE;
    TRY_CUDA(cudaSetDevice(ctx->device));
    int launches = 0;
    TRY(ensure_degree_hist(ctx, &launches));
    TRY_CUDA(cudaStreamSynchronize(ctx->stream));
    if (hist_dev) *hist_dev = (const int64_t*)ctx->deg_hist.p;
    if (max_degree_out) *max_degree_out = ctx->max_degree;
    return TCRNET_OK;
}

int tcrnet_neighbor_degree(tcrnet_ctx* ctx, const int64_t** nn_sum_dev, const int64_t** class_sum_dev,
                           const double** knn_dev) {
    if (!ctx) return TCRNET_ERR_ARG;
    if (!ctx->built) return TCRNET_ERR_STATE;
    TRY_CUDA(cudaSetDevice(ctx->device));
    cudaStream_t s = ctx->stream;
    int launches = 0;
    TRY(ensure_degree_hist(ctx, &launches));
    if (!ctx->have_nn) {
        const int32_t hist_len = ctx->max_degree + 1;
        TRY(dev_reserve(ctx, ctx->nn_sum, sizeof(unsigned long long) * (size_t)ctx->n));
        TRY(dev_reserve(ctx, ctx->class_sum, sizeof(unsigned long long) * (size_t)hist_len));
        TRY(dev_reserve(ctx, ctx->knn, sizeof(double) * (size_t)hist_len));
        TRY_CUDA(cudaMemsetAsync(ctx->nn_sum.p, 0, sizeof(unsigned long long) * (size_t)ctx->n, s));
        TRY_CUDA(cudaMemsetAsync(ctx->class_sum.p, 0, sizeof(unsigned long long) * (size_t)hist_len, s));
        TRY_CUDA(launch_neighbor_degree((const int64_t*)ctx->row_ptr.p, (const int32_t*)ctx->col.p,
                                        (const int32_t*)ctx->deg.p, ctx->n, (const unsigned long long*)ctx->deg_hist.p,
                                        hist_len, (unsigned long long*)ctx->nn_sum.p,
                                        (unsigned long long*)ctx->class_sum.p, (double*)ctx->knn.p, s, &launches));
        ctx->have_nn = true;
    }
    TRY_CUDA(cudaStreamSynchronize(s));
    if (nn_sum_dev) *nn_sum_dev = (const int64_t*)ctx->nn_sum.p;
    if (class_sum_dev) *class_sum_dev = (const int64_t*)ctx->class_sum.p;
    if (knn_dev) *knn_dev = (const double*)ctx->knn.p;
    return TCRNET_OK;
}

int tcrnet_components(tcrnet_ctx* ctx, const int32_t** label_dev, const int32_t** comp_size_dev,
                      int64_t* n_components_out, int64_t* lcc_out) {
    if (!ctx) return TCRNET_ERR_ARG;
    if (!ctx->built) return TCRNET_ERR_STATE;
    TRY_CUDA(cudaSetDevice(ctx->device));
    int launches = 0;
    TRY(ensure_components(ctx, &launches));
    if (label_dev) *label_dev = (const int32_t*)ctx->cc_label.p;
    if (comp_size_dev) *comp_size_dev = (const int32_t*)ctx->cc_size.p;
    if (n_components_out) *n_components_out = ctx->n_components;
    if (lcc_out) *lcc_out = ctx->lcc;
    return TCRNET_OK;
}

int tcrnet_percolation(tcrnet_ctx* ctx, const int32_t* removal_rank, const int64_t* n_removed, int32_t n_steps,
                       int64_t* lcc_out, double* lcc_norm1_out, double* lcc_norm2_out, int64_t* deg_hist_out) {
    if (!ctx || !removal_rank || n_steps < 0 || (n_steps > 0 && !n_removed)) return TCRNET_ERR_ARG;
    if (!ctx->built) return TCRNET_ERR_STATE;
    const int64_t n = ctx->n;
    for (int32_t k = 0; k < n_steps; ++k)
        if (n_removed[k] < 0 || n_removed[k] > n) return TCRNET_ERR_ARG;
    TRY_CUDA(cudaSetDevice(ctx->device));
    cudaStream_t s = ctx->stream;
    int launches = 0;

    // the removal order: copy, check that it is a permutation
    const size_t seen_bytes = sizeof(uint32_t) * (size_t)((n + 31) / 32);
    TRY(dev_reserve(ctx, ctx->obs_ctrl, sizeof(ObsCtrl)));
    TRY(dev_reserve(ctx, ctx->perc_rank, sizeof(int32_t) * (size_t)n));
    TRY(dev_reserve(ctx, ctx->perc_seen, seen_bytes));
    TRY_CUDA(cudaMemcpyAsync(ctx->perc_rank.p, removal_rank, sizeof(int32_t) * (size_t)n, cudaMemcpyHostToDevice, s));
    TRY_CUDA(cudaMemsetAsync(ctx->perc_seen.p, 0, seen_bytes, s));
    TRY_CUDA(cudaMemsetAsync(&d_obs(ctx)->flag, 0, sizeof(uint32_t), s));
    TRY_CUDA(launch_check_permutation((const int32_t*)ctx->perc_rank.p, n, (uint32_t*)ctx->perc_seen.p,
                                      &d_obs(ctx)->flag, s, &launches));
    ObsCtrl h{};
    TRY(fetch_ctrl(ctx, &h));  // also ends the borrow of removal_rank
    if (h.flag) return TCRNET_ERR_ARG;

    TRY(ensure_components(ctx, &launches));  // LCC at p = 0 for Eq. 13
    int32_t hist_len = 0;
    if (deg_hist_out) {
        TRY(ensure_degree_hist(ctx, &launches));
        hist_len = ctx->max_degree + 1;
    }
    if (n_steps == 0) return TCRNET_OK;

    // per step: [k] = LCC, [n_steps + k] = number of components (not reported)
    const size_t res_bytes = sizeof(unsigned long long) * 2 * (size_t)n_steps;
    const size_t hist_bytes = sizeof(unsigned long long) * (size_t)hist_len * (size_t)n_steps;
    TRY(dev_reserve(ctx, ctx->perc_lcc, res_bytes));
    TRY(dev_reserve(ctx, ctx->cc_parent, sizeof(int32_t) * (size_t)n));
    TRY(dev_reserve(ctx, ctx->perc_deg, sizeof(int32_t) * (size_t)n));  // degrees inside the induced subgraph
    TRY_CUDA(cudaMemsetAsync(ctx->perc_lcc.p, 0, res_bytes, s));
    int32_t* sub_deg = nullptr;
    DevBuf& count = ctx->perc_seen;  // reuse: int32[n] component counters of a step
    TRY(dev_reserve(ctx, count, sizeof(int32_t) * (size_t)n));
    if (deg_hist_out) {
        TRY(dev_reserve(ctx, ctx->perc_hist, hist_bytes));
        TRY_CUDA(cudaMemsetAsync(ctx->perc_hist.p, 0, hist_bytes, s));
        sub_deg = (int32_t*)ctx->perc_deg.p;
    }
    unsigned long long* res = (unsigned long long*)ctx->perc_lcc.p;
    for (int32_t k = 0; k < n_steps; ++k) {
        const int32_t thr = (int32_t)n_removed[k];
        TRY_CUDA(launch_components((const int64_t*)ctx->row_ptr.p, (const int32_t*)ctx->col.p, n,
                                   (const int32_t*)ctx->perc_rank.p, thr, (int32_t*)ctx->cc_parent.p, (int32_t*)count.p,
                                   nullptr, sub_deg, res + k, res + n_steps + k, s, &launches));
        if (sub_deg)
            TRY_CUDA(launch_degree_hist(sub_deg, n, (const int32_t*)ctx->perc_rank.p, thr,
                                        (unsigned long long*)ctx->perc_hist.p + (size_t)k * hist_len, s, &launches));
    }
    std::vector<unsigned long long> lcc((size_t)n_steps);
    TRY_CUDA(cudaMemcpyAsync(lcc.data(), res, sizeof(unsigned long long) * (size_t)n_steps, cudaMemcpyDeviceToHost, s));
    if (deg_hist_out)
        TRY_CUDA(cudaMemcpyAsync(deg_hist_out, ctx->perc_hist.p, hist_bytes, cudaMemcpyDeviceToHost, s));
    TRY_CUDA(cudaStreamSynchronize(s));
    // Eq. 12 / Eq. 13: integer results -> two IEEE divisions each
    const double norm1_at_0 = n > 0 ? (double)ctx->lcc / (double)n : 0.0;
    for (int32_t k = 0; k < n_steps; ++k) {
        const int64_t left = n - n_removed[k];
        const double n1 = left > 0 ? (double)(int64_t)lcc[k] / (double)left : 0.0;
        if (lcc_out) lcc_out[k] = (int64_t)lcc[k];
        if (lcc_norm1_out) lcc_norm1_out[k] = n1;
        if (lcc_norm2_out) lcc_norm2_out[k] = norm1_at_0 > 0.0 ? n1 / norm1_at_0 : 0.0;
    }
    return TCRNET_OK;
}

}  // extern "C"

// Network observables on the CSR (section II.G-II.J, Fig. 2(f)-(h)):
// degree distribution, average neighbour degree (Eq. 9), connected components / LCC, and the
// per-step work of the site-percolation sweep.  All of it is HBM/L2-bound streaming over
// row_ptr (8 B/node), col (4 B/edge), deg (4 B/node) plus L2 atomics; nothing here is a contraction.
//
// Components: lock-free union-find over the strict-upper-triangle edges.  Hooking always puts the
// LARGER root under the SMALLER one (atomicCAS on the larger root), so parent[x] <= x holds at all
// times (no cycles) and the final root of a component is its smallest node id - the unique label
// the oracle's breadth-first search yields.  find() uses path halving with plain stores (a stale
// parent is still an ancestor in the same tree, so races only cost extra hops); parent reads bypass
// L1 (ld.global.cg) so that a CAS loser sees the winner's update.
#include "launch.cuh"
#include "tcrnet_internal.h"

namespace tcrnet {
namespace {

constexpr int kHistSmem = 1024;  // degree classes accumulated in shared memory; larger degrees go to L2

__device__ __forceinline__ bool node_alive(const int32_t* __restrict__ rank, int32_t threshold, int64_t u) {
    return rank == nullptr || rank[u] >= threshold;
}

// ---- degree distribution -------------------------------------------------------------------

__global__ void __launch_bounds__(256) k_max_degree(const int32_t* __restrict__ deg, int64_t n, int32_t* out) {
    grid_dependency_wait();
    int32_t m = 0;
    for (int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; u < n; u += (int64_t)gridDim.x * blockDim.x)
        m = max(m, deg[u]);
    m = __reduce_max_sync(0xffffffffu, m);
    if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(out, m);
}

// hist[d] += #{u alive : deg[u] = d}.  `deg` is the degree to count (full network or the induced
// subgraph of a percolation step); rank/threshold select the alive nodes (rank == NULL: all).
__global__ void __launch_bounds__(256) k_degree_hist(const int32_t* __restrict__ deg, int64_t n,
                                                    const int32_t* __restrict__ rank, int32_t threshold,
                                                    unsigned long long* __restrict__ hist) {
    grid_dependency_wait();
    __shared__ uint32_t sh[kHistSmem];
    for (int i = threadIdx.x; i < kHistSmem; i += blockDim.x) sh[i] = 0u;
    __syncthreads();
    for (int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; u < n; u += (int64_t)gridDim.x * blockDim.x) {
        if (!node_alive(rank, threshold, u)) continue;
        const int32_t d = deg[u];
        if (d < kHistSmem) atomicAdd(&sh[d], 1u);
        else atomicAdd(&hist[d], 1ull);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < kHistSmem; i += blockDim.x)
        if (sh[i]) atomicAdd(&hist[i], (unsigned long long)sh[i]);
}

// ---- average neighbour degree (Eq. 9) ------------------------------------------------------

// One thread per row u of the upper triangle: every edge (u, v) adds d(v) to nn_sum[u] and d(u) to
// nn_sum[v] (A is symmetric).
__global__ void __launch_bounds__(256) k_nn_sum(const int64_t* __restrict__ row_ptr, const int32_t* __restrict__ col,
                                               const int32_t* __restrict__ deg, int64_t n,
                                               unsigned long long* __restrict__ nn_sum) {
    grid_dependency_wait();
    const int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= n) return;
    const int64_t b = row_ptr[u], e = row_ptr[u + 1];
    if (b == e) return;
    const unsigned long long du = (unsigned long long)deg[u];
    unsigned long long acc = 0ull;
    for (int64_t k = b; k < e; ++k) {
        const int32_t v = col[k];
        acc += (unsigned long long)deg[v];
        atomicAdd(&nn_sum[v], du);
    }
    atomicAdd(&nn_sum[u], acc);
}

__global__ void __launch_bounds__(256) k_class_sum(const int32_t* __restrict__ deg,
                                                  const unsigned long long* __restrict__ nn_sum, int64_t n,
                                                  unsigned long long* __restrict__ class_sum) {
    grid_dependency_wait();
    __shared__ unsigned long long sh[kHistSmem];
    for (int i = threadIdx.x; i < kHistSmem; i += blockDim.x) sh[i] = 0ull;
    __syncthreads();
    for (int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; u < n; u += (int64_t)gridDim.x * blockDim.x) {
        const int32_t d = deg[u];
        const unsigned long long s = nn_sum[u];
        if (s == 0ull) continue;
        if (d < kHistSmem) atomicAdd(&sh[d], s);
        else atomicAdd(&class_sum[d], s);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < kHistSmem; i += blockDim.x)
        if (sh[i]) atomicAdd(&class_sum[i], sh[i]);
}

// <d_nn>(d) = class_sum[d] / (d * hist[d]): one IEEE division of two exactly converted integers.
__global__ void __launch_bounds__(256) k_knn(const unsigned long long* __restrict__ class_sum,
                                            const unsigned long long* __restrict__ hist, int32_t hist_len,
                                            double* __restrict__ knn) {
    grid_dependency_wait();
    const int d = blockIdx.x * blockDim.x + threadIdx.x;
    if (d >= hist_len) return;
    double v = 0.0;
    if (d > 0 && hist[d] > 0ull) v = __ddiv_rn((double)(long long)class_sum[d], (double)((long long)d * (long long)hist[d]));
    knn[d] = v;
}

// ---- connected components ------------------------------------------------------------------

__device__ __forceinline__ int32_t cc_find(int32_t* parent, int32_t x) {
    int32_t p = __ldcg(parent + x);
    while (p != x) {
        const int32_t gp = __ldcg(parent + p);
        if (gp != p) parent[x] = gp;  // path halving
        x = p;
        p = gp;
    }
    return x;
}

__device__ __forceinline__ void cc_unite(int32_t* parent, int32_t a, int32_t b) {
    int32_t ra = cc_find(parent, a), rb = cc_find(parent, b);
    while (ra != rb) {
        if (ra < rb) {
            const int32_t t = ra;
            ra = rb;
            rb = t;
        }
        // ra > rb: hook ra under rb if ra is still a root
        const int32_t old = atomicCAS(parent + ra, ra, rb);
        if (old == ra) return;
        ra = cc_find(parent, old);
        rb = cc_find(parent, rb);
    }
}

// parent[u] = u, count[u] = 0 (dead nodes too: they are simply never hooked or counted)
__global__ void __launch_bounds__(256) k_cc_init(int64_t n, int32_t* __restrict__ parent, int32_t* __restrict__ count,
                                                int32_t* __restrict__ sub_deg) {
    grid_dependency_wait();
    const int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= n) return;
    parent[u] = (int32_t)u;
    count[u] = 0;
    if (sub_deg) sub_deg[u] = 0;
}

// One thread per row: unite the endpoints of every edge whose two ends are alive; optionally count
// the degrees inside the induced subgraph.
__global__ void __launch_bounds__(256) k_cc_hook(const int64_t* __restrict__ row_ptr, const int32_t* __restrict__ col,
                                                int64_t n, const int32_t* __restrict__ rank, int32_t threshold,
                                                int32_t* parent, int32_t* __restrict__ sub_deg) {
    grid_dependency_wait();
    const int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= n || !node_alive(rank, threshold, u)) return;
    const int64_t b = row_ptr[u], e = row_ptr[u + 1];
    int32_t mine = 0;
    for (int64_t k = b; k < e; ++k) {
        const int32_t v = col[k];
        if (!node_alive(rank, threshold, v)) continue;
        cc_unite(parent, (int32_t)u, v);
        if (sub_deg) {
            ++mine;
            atomicAdd(&sub_deg[v], 1);
        }
    }
    if (sub_deg && mine) atomicAdd(&sub_deg[u], mine);
}

// label[u] = root of u (dead: -1); count[root] += 1 (aggregated over the lanes of a warp that share a
// root); *lcc = max over all partial counts = size of the largest component; *n_comp += #roots.
__global__ void __launch_bounds__(256) k_cc_label(int64_t n, const int32_t* __restrict__ rank, int32_t threshold,
                                                 int32_t* parent, int32_t* __restrict__ label,
                                                 int32_t* __restrict__ count, unsigned long long* lcc,
                                                 unsigned long long* n_comp) {
    grid_dependency_wait();
    const int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool alive = u < n && node_alive(rank, threshold, u);
    int32_t root = -1;
    if (alive) root = cc_find(parent, (int32_t)u);
    if (u < n && label) label[u] = root;
    const uint32_t peers = __match_any_sync(0xffffffffu, root);
    int32_t seen = 0;
    if (alive && (int)(__ffs((int)peers) - 1) == (int)(threadIdx.x & 31)) {
        const int32_t c = __popc(peers);
        seen = atomicAdd(&count[root], c) + c;
    }
    seen = __reduce_max_sync(0xffffffffu, seen);
    const uint32_t roots = __ballot_sync(0xffffffffu, alive && root == (int32_t)u);
    if ((threadIdx.x & 31) == 0) {
        if (seen > 0) atomicMax(lcc, (unsigned long long)seen);
        if (roots) atomicAdd(n_comp, (unsigned long long)__popc(roots));
    }
}

__global__ void __launch_bounds__(256) k_cc_sizes(int64_t n, const int32_t* __restrict__ label,
                                                 const int32_t* __restrict__ count, int32_t* __restrict__ comp_size) {
    grid_dependency_wait();
    const int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= n) return;
    const int32_t r = label[u];
    comp_size[u] = r >= 0 ? count[r] : 0;
}

// ---- removal order validation ----------------------------------------------------------------

// *flag |= 1 unless rank is a permutation of 0..n-1 (seen must be zeroed)
__global__ void __launch_bounds__(256) k_check_permutation(const int32_t* __restrict__ rank, int64_t n,
                                                          uint32_t* __restrict__ seen, uint32_t* flag) {
    grid_dependency_wait();
    const int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= n) return;
    const int32_t r = rank[u];
    if (r < 0 || (int64_t)r >= n) {
        atomicOr(flag, 1u);
        return;
    }
    const uint32_t bit = 1u << (r & 31);
    if (atomicOr(&seen[r >> 5], bit) & bit) atomicOr(flag, 1u);
}

unsigned grid_for(int64_t n) { return (unsigned)((n + 255) / 256); }
unsigned grid_capped(int64_t n) {
    int64_t b = (n + 255) / 256;
    if (b > device_sm_count() * 8) b = device_sm_count() * 8;
    return (unsigned)(b > 0 ? b : 1);
}

}  // namespace

cudaError_t launch_max_degree(const int32_t* deg, int64_t n, int32_t* out, cudaStream_t s, int* launches) {
    launch_dep(k_max_degree, grid_capped(n), 256, 0, s, deg, n, out);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_degree_hist(const int32_t* deg, int64_t n, const int32_t* rank, int32_t threshold,
                               unsigned long long* hist, cudaStream_t s, int* launches) {
    launch_dep(k_degree_hist, grid_capped(n), 256, 0, s, deg, n, rank, threshold, hist);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_neighbor_degree(const int64_t* row_ptr, const int32_t* col, const int32_t* deg, int64_t n,
                                   const unsigned long long* hist, int32_t hist_len, unsigned long long* nn_sum,
                                   unsigned long long* class_sum, double* knn, cudaStream_t s, int* launches) {
    launch_dep(k_nn_sum, grid_for(n), 256, 0, s, row_ptr, col, deg, n, nn_sum);
    launch_dep(k_class_sum, grid_capped(n), 256, 0, s, deg, nn_sum, n, class_sum);
    launch_dep(k_knn, grid_for(hist_len), 256, 0, s, class_sum, hist, hist_len, knn);
    *launches += 3;
    return cudaGetLastError();
}

cudaError_t launch_components(const int64_t* row_ptr, const int32_t* col, int64_t n, const int32_t* rank,
                              int32_t threshold, int32_t* parent, int32_t* count, int32_t* label, int32_t* sub_deg,
                              unsigned long long* lcc, unsigned long long* n_comp, cudaStream_t s, int* launches) {
    launch_dep(k_cc_init, grid_for(n), 256, 0, s, n, parent, count, sub_deg);
    launch_dep(k_cc_hook, grid_for(n), 256, 0, s, row_ptr, col, n, rank, threshold, parent, sub_deg);
    launch_dep(k_cc_label, grid_for(n), 256, 0, s, n, rank, threshold, parent, label, count, lcc, n_comp);
    *launches += 3;
    return cudaGetLastError();
}

cudaError_t launch_component_sizes(int64_t n, const int32_t* label, const int32_t* count, int32_t* comp_size,
                                   cudaStream_t s, int* launches) {
    launch_dep(k_cc_sizes, grid_for(n), 256, 0, s, n, label, count, comp_size);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_check_permutation(const int32_t* rank, int64_t n, uint32_t* seen, uint32_t* flag, cudaStream_t s,
                                     int* launches) {
    launch_dep(k_check_permutation, grid_for(n), 256, 0, s, rank, n, seen, flag);
    *launches += 1;
    return cudaGetLastError();
}

}  // namespace tcrnet

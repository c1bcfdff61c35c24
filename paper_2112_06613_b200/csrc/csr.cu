// Step A6, second half: sorted edge keys -> CSR of the strict upper triangle + degrees
// (PAPER.md:301-318 adjacency matrix, PAPER.md:224 degree d(u) = sum_v A_uv).
//
//   row_ptr[r] = number of edges whose first index is < r = lower bound of (r << 32) in the
//                sorted keys: one binary search per row, no serial gap filling, no skew.
//   col[e]     = second index of edge e.
//   deg[u]     = (row_ptr[u+1] - row_ptr[u])  [edges (u, v>u)]  +  #{e : col[e] = u}  [edges (w<u, u)].
// HBM-bound: 8 B read + 4 B write per edge, 12 B written per node, plus one L2 atomic per edge.
#include "tcrnet_internal.h"

namespace tcrnet {
namespace {

__global__ void __launch_bounds__(256) k_row_ptr(const unsigned long long* __restrict__ keys, int64_t n_edges,
                                                int64_t n, int64_t* __restrict__ row_ptr) {
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r > n) return;
    const unsigned long long want = (unsigned long long)r << 32;
    int64_t lo = 0, hi = n_edges;  // first e with keys[e] >= want
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (keys[mid] < want) lo = mid + 1; else hi = mid;
    }
    row_ptr[r] = lo;
}

__global__ void __launch_bounds__(256) k_deg_upper(const int64_t* __restrict__ row_ptr, int64_t n,
                                                  int32_t* __restrict__ deg) {
    const int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (u < n) deg[u] = (int32_t)(row_ptr[u + 1] - row_ptr[u]);
}

__global__ void __launch_bounds__(256) k_col_deg_lower(const unsigned long long* __restrict__ keys, int64_t n_edges,
                                                      int32_t* __restrict__ col, int32_t* __restrict__ deg) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_edges;
         e += (int64_t)gridDim.x * blockDim.x) {
        const uint32_t v = (uint32_t)keys[e];
        col[e] = (int32_t)v;
        atomicAdd(&deg[v], 1);
    }
}

}  // namespace

cudaError_t launch_csr(const unsigned long long* sorted_keys, int64_t n_edges, int64_t n, int64_t* row_ptr,
                       int32_t* col, int32_t* deg, cudaStream_t s, int* launches) {
    k_row_ptr<<<(unsigned)((n + 1 + 255) / 256), 256, 0, s>>>(sorted_keys, n_edges, n, row_ptr);
    k_deg_upper<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(row_ptr, n, deg);
    *launches += 2;
    if (n_edges > 0) {
        int64_t blocks = (n_edges + 255) / 256;
        if (blocks > 148 * 16) blocks = 148 * 16;
        k_col_deg_lower<<<(unsigned)blocks, 256, 0, s>>>(sorted_keys, n_edges, col, deg);
        *launches += 1;
    }
    return cudaGetLastError();
}

}  // namespace tcrnet

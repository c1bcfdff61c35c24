// Distance labels of the final edges and threshold restriction (one build at
// the largest threshold serves every smaller one - PAPER.md:105 / Fig. 2(i) sweeps l_max), plus
// the key validation of tcrnet_assemble.
//
// The distance kernels decide "lev <= l_max" for ~10^11 pairs and keep ~10^6..10^7 of them; the
// labels are computed afterwards for the kept edges only: one thread per edge, the Myers/Hyyro
// column recurrence on one word, the match mask of each column derived from the two bit-plane rows
// (Eq = AND over the five planes of "plane of a agrees with bit k of the text residue": five selects),
// so an edge costs two 32-byte rows and ~25 instructions per column.  The first index of every edge
// is written once per CSR by k_edge_rows (one thread per row) instead of a binary search per edge.
// HBM/L2-bound: 2 plane rows read and 1 byte written per edge.
#include "launch.cuh"
#include "planes.cuh"
#include "tcrnet_internal.h"

namespace tcrnet {
namespace {

__global__ void __launch_bounds__(256) k_inverse_perm(const int32_t* __restrict__ perm, int64_t n,
                                                     int32_t* __restrict__ inv) {
    grid_dependency_wait();
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) inv[perm[s]] = (int32_t)s;
}

// edge_row[e] = first index of edge e (the row r with row_ptr[r] <= e < row_ptr[r+1])
__global__ void __launch_bounds__(256) k_edge_rows(const int64_t* __restrict__ row_ptr, int64_t n,
                                                  int32_t* __restrict__ edge_row) {
    grid_dependency_wait();
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    const int64_t b = row_ptr[r], e = row_ptr[r + 1];
    for (int64_t k = b; k < e; ++k) edge_row[k] = (int32_t)r;
}

// lev(a, b) column by column: Pv / Mv are the +1 / -1 vertical deltas of the current DP column,
// the "| 1" is the boundary D[0][j] = j; |a| = m <= bits of W.
template <typename W>
__device__ __forceinline__ int lev_planes(const PlaneRow<W>& A, const PlaneRow<W>& B) {
    const int m = A.len, n = B.len;
    if (m == 0) return n;
    const W low_m = m >= (int)(8 * sizeof(W)) ? ~W(0) : ((W(1) << m) - W(1));
    W Pv = low_m, Mv = W(0);
    for (int j = 0; j < n; ++j) {
        W Eq = low_m;
#pragma unroll
        for (int k = 0; k < 5; ++k) Eq &= ((B.p[k] >> j) & W(1)) ? A.p[k] : ~A.p[k];
        const W D0 = ((((Eq & Pv) + Pv) ^ Pv) | Eq) | Mv;
        const W Hp = Mv | ~(D0 | Pv);
        const W Hn = Pv & D0;
        const W Hp1 = (Hp << 1) | W(1);
        Pv = (Hn << 1) | ~(D0 | Hp1);
        Mv = D0 & Hp1;
    }
    const W pm = Pv & low_m, mm = Mv & low_m;
    return n + (sizeof(W) == 8 ? __popcll((unsigned long long)pm) - __popcll((unsigned long long)mm)
                               : __popc((uint32_t)pm) - __popc((uint32_t)mm));
}

template <typename W>
__global__ void __launch_bounds__(256) k_edge_distances(const int32_t* __restrict__ edge_row,
                                                       const int32_t* __restrict__ col, int64_t n_edges,
                                                       const int32_t* __restrict__ inv_perm,
                                                       const void* __restrict__ planes, uint8_t* __restrict__ dist) {
    grid_dependency_wait();
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_edges) return;
    const PlaneRow<W> A = load_planes<W>(planes, inv_perm[edge_row[e]]);
    const PlaneRow<W> B = load_planes<W>(planes, inv_perm[col[e]]);
    dist[e] = (uint8_t)lev_planes<W>(A, B);
}

__global__ void __launch_bounds__(256) k_restrict_flags(const uint8_t* __restrict__ dist, int64_t n_edges, int l_max,
                                                       uint32_t* __restrict__ flags) {
    grid_dependency_wait();
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < n_edges) flags[e] = (int)dist[e] <= l_max ? 1u : 0u;
}

__global__ void __launch_bounds__(256) k_restrict_compact(const int32_t* __restrict__ edge_row,
                                                         const int32_t* __restrict__ col,
                                                         const uint8_t* __restrict__ dist, int64_t n_edges,
                                                         const uint32_t* __restrict__ flags,
                                                         const uint32_t* __restrict__ pos,
                                                         unsigned long long* __restrict__ keys_out,
                                                         uint8_t* __restrict__ dist_out) {
    grid_dependency_wait();
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_edges || !flags[e]) return;
    const unsigned long long u = (unsigned long long)(uint32_t)edge_row[e];
    keys_out[pos[e]] = (u << 32) | (uint32_t)col[e];
    dist_out[pos[e]] = dist[e];
}

__global__ void __launch_bounds__(256) k_validate_keys(const unsigned long long* __restrict__ keys, int64_t n_keys,
                                                      int64_t n, uint32_t* __restrict__ flag) {
    grid_dependency_wait();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool bad = false;
    if (i < n_keys) {
        const unsigned long long k = keys[i];
        const unsigned long long u = k >> 32, v = k & 0xffffffffull;
        bad = u >= v || v >= (unsigned long long)n;
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(flag, 1u);
}

inline unsigned grid_for(int64_t n) { return (unsigned)((n + 255) / 256); }

}  // namespace

cudaError_t launch_inverse_perm(const int32_t* perm, int64_t n, int32_t* inv, cudaStream_t s, int* launches) {
    launch_dep(k_inverse_perm, grid_for(n), 256, 0, s, perm, n, inv);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_edge_rows(const int64_t* row_ptr, int64_t n, int32_t* edge_row, cudaStream_t s, int* launches) {
    if (n <= 0) return cudaSuccess;
    launch_dep(k_edge_rows, grid_for(n), 256, 0, s, row_ptr, n, edge_row);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_edge_distances(const int32_t* edge_row, const int32_t* col, int64_t n_edges, const int32_t* inv_perm,
                                  const void* planes, bool wide_planes, uint8_t* dist, cudaStream_t s, int* launches) {
    if (n_edges <= 0) return cudaSuccess;
    if (wide_planes) launch_dep(k_edge_distances<uint64_t>, grid_for(n_edges), 256, 0, s, edge_row, col, n_edges,
                                inv_perm, planes, dist);
    else launch_dep(k_edge_distances<uint32_t>, grid_for(n_edges), 256, 0, s, edge_row, col, n_edges, inv_perm,
                    planes, dist);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_restrict_flags(const uint8_t* dist, int64_t n_edges, int l_max, uint32_t* flags, cudaStream_t s,
                                  int* launches) {
    if (n_edges <= 0) return cudaSuccess;
    launch_dep(k_restrict_flags, grid_for(n_edges), 256, 0, s, dist, n_edges, l_max, flags);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_restrict_compact(const int32_t* edge_row, const int32_t* col, const uint8_t* dist,
                                    int64_t n_edges, const uint32_t* flags, const uint32_t* pos,
                                    unsigned long long* keys_out, uint8_t* dist_out, cudaStream_t s, int* launches) {
    if (n_edges <= 0) return cudaSuccess;
    launch_dep(k_restrict_compact, grid_for(n_edges), 256, 0, s, edge_row, col, dist, n_edges, flags, pos, keys_out,
               dist_out);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_validate_keys(const unsigned long long* keys, int64_t n_keys, int64_t n, uint32_t* flag,
                                 cudaStream_t s, int* launches) {
    if (n_keys <= 0) return cudaSuccess;
    launch_dep(k_validate_keys, grid_for(n_keys), 256, 0, s, keys, n_keys, n, flag);
    *launches += 1;
    return cudaGetLastError();
}

}  // namespace tcrnet

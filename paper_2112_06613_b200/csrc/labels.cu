// Distance labels of the final edges and threshold restriction (one build at
// the largest threshold serves every smaller one - PAPER.md:105 / Fig. 2(i) sweeps l_max), plus
// the key validation of tcrnet_assemble.
//
// The distance kernels decide "lev <= l_max" for ~10^11 pairs and keep ~10^6..10^7 of them; the
// labels are computed afterwards for the kept edges only (one thread per edge, the same
// Myers/Hyyro column recurrence on a 64-bit word with the match mask of each column derived on
// the fly from the pattern bytes), which costs microseconds and needs no room in the edge keys.
// HBM/L2-bound: 2 pattern rows (<= 128 B) read and 1 byte written per edge.
#include "tcrnet_internal.h"

namespace tcrnet {
namespace {

__global__ void __launch_bounds__(256) k_inverse_perm(const int32_t* __restrict__ perm, int64_t n,
                                                     int32_t* __restrict__ inv) {
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) inv[perm[s]] = (int32_t)s;
}

// first index of edge e = the row r with row_ptr[r] <= e < row_ptr[r+1]
__device__ __forceinline__ int64_t row_of_edge(const int64_t* __restrict__ row_ptr, int64_t n, int64_t e) {
    int64_t lo = 0, hi = n;  // invariant: row_ptr[lo] <= e < row_ptr[hi]
    while (hi - lo > 1) {
        const int64_t mid = (lo + hi) >> 1;
        if (row_ptr[mid] <= e) lo = mid; else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ int row_length(const uint8_t* row, int pat_stride) {
    int len = 0;
    while (len < pat_stride && row[len] != 0xffu) ++len;
    return len;
}

// lev(a, b) for |a| = m <= 64: Pv / Mv are the +1 / -1 vertical deltas of the current DP column
// (PAPER.md:277-293 computed column by column; the "| 1" is the boundary D[0][j] = j).
__device__ int lev64(const uint8_t* a, int m, const uint8_t* b, int n) {
    if (m == 0) return n;
    const unsigned long long low_m = m >= 64 ? ~0ull : ((1ull << m) - 1ull);
    unsigned long long Pv = low_m, Mv = 0ull;
    for (int j = 0; j < n; ++j) {
        const uint8_t c = b[j];
        unsigned long long Eq = 0ull;
        for (int i = 0; i < m; ++i) Eq |= (unsigned long long)(a[i] == c) << i;
        const unsigned long long D0 = ((((Eq & Pv) + Pv) ^ Pv) | Eq) | Mv;
        const unsigned long long Hp = Mv | ~(D0 | Pv);
        const unsigned long long Hn = Pv & D0;
        const unsigned long long Hp1 = (Hp << 1) | 1ull;
        Pv = (Hn << 1) | ~(D0 | Hp1);
        Mv = D0 & Hp1;
    }
    return n + __popcll(Pv & low_m) - __popcll(Mv & low_m);
}

__global__ void __launch_bounds__(256) k_edge_distances(const int64_t* __restrict__ row_ptr,
                                                       const int32_t* __restrict__ col, int64_t n, int64_t n_edges,
                                                       const int32_t* __restrict__ inv_perm,
                                                       const uint8_t* __restrict__ pat, int pat_stride,
                                                       uint8_t* __restrict__ dist) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_edges) return;
    const int64_t u = row_of_edge(row_ptr, n, e);
    const int64_t v = col[e];
    const uint8_t* a = pat + (size_t)inv_perm[u] * pat_stride;
    const uint8_t* b = pat + (size_t)inv_perm[v] * pat_stride;
    dist[e] = (uint8_t)lev64(a, row_length(a, pat_stride), b, row_length(b, pat_stride));
}

__global__ void __launch_bounds__(256) k_restrict_flags(const uint8_t* __restrict__ dist, int64_t n_edges, int l_max,
                                                       uint32_t* __restrict__ flags) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < n_edges) flags[e] = (int)dist[e] <= l_max ? 1u : 0u;
}

__global__ void __launch_bounds__(256) k_restrict_compact(const int64_t* __restrict__ row_ptr,
                                                         const int32_t* __restrict__ col,
                                                         const uint8_t* __restrict__ dist, int64_t n, int64_t n_edges,
                                                         const uint32_t* __restrict__ flags,
                                                         const uint32_t* __restrict__ pos,
                                                         unsigned long long* __restrict__ keys_out,
                                                         uint8_t* __restrict__ dist_out) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_edges || !flags[e]) return;
    const unsigned long long u = (unsigned long long)row_of_edge(row_ptr, n, e);
    keys_out[pos[e]] = (u << 32) | (uint32_t)col[e];
    dist_out[pos[e]] = dist[e];
}

__global__ void __launch_bounds__(256) k_validate_keys(const unsigned long long* __restrict__ keys, int64_t n_keys,
                                                      int64_t n, uint32_t* __restrict__ flag) {
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
    k_inverse_perm<<<grid_for(n), 256, 0, s>>>(perm, n, inv);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_edge_distances(const int64_t* row_ptr, const int32_t* col, int64_t n, int64_t n_edges,
                                  const int32_t* inv_perm, const uint8_t* pat, int pat_stride, uint8_t* dist,
                                  cudaStream_t s, int* launches) {
    if (n_edges <= 0) return cudaSuccess;
    k_edge_distances<<<grid_for(n_edges), 256, 0, s>>>(row_ptr, col, n, n_edges, inv_perm, pat, pat_stride, dist);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_restrict_flags(const uint8_t* dist, int64_t n_edges, int l_max, uint32_t* flags, cudaStream_t s,
                                  int* launches) {
    if (n_edges <= 0) return cudaSuccess;
    k_restrict_flags<<<grid_for(n_edges), 256, 0, s>>>(dist, n_edges, l_max, flags);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_restrict_compact(const int64_t* row_ptr, const int32_t* col, const uint8_t* dist, int64_t n,
                                    int64_t n_edges, const uint32_t* flags, const uint32_t* pos,
                                    unsigned long long* keys_out, uint8_t* dist_out, cudaStream_t s, int* launches) {
    if (n_edges <= 0) return cudaSuccess;
    k_restrict_compact<<<grid_for(n_edges), 256, 0, s>>>(row_ptr, col, dist, n, n_edges, flags, pos, keys_out,
                                                         dist_out);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_validate_keys(const unsigned long long* keys, int64_t n_keys, int64_t n, uint32_t* flag,
                                 cudaStream_t s, int* launches) {
    if (n_keys <= 0) return cudaSuccess;
    k_validate_keys<<<grid_for(n_keys), 256, 0, s>>>(keys, n_keys, n, flag);
    *launches += 1;
    return cudaGetLastError();
}

}  // namespace tcrnet

// Step A6, second half: sorted edge keys -> CSR of the strict upper triangle + degrees
// (PAPER.md:301-318 adjacency matrix, PAPER.md:224 degree d(u) = sum_v A_uv).
//
//   row_ptr[r] = number of edges whose first index is < r = lower bound of (r << 32) in the
//                sorted keys: one binary search per row, no serial gap filling, no skew.
//   col[e]     = second index of edge e.
//   deg[u]     = (row_ptr[u+1] - row_ptr[u])  [edges (u, v>u)]  +  #{e : col[e] = u}  [edges (w<u, u)].
// HBM-bound: 8 B read + 4 B write per edge, 12 B written per node, plus one L2 atomic per edge.
#include <algorithm>

#include "launch.cuh"
#include "tcrnet_internal.h"

namespace tcrnet {
namespace {

__global__ void __launch_bounds__(256) k_row_ptr(const unsigned long long* __restrict__ keys, int64_t n_edges,
                                                int64_t n, int64_t* __restrict__ row_ptr) {
    grid_dependency_wait();
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
    grid_dependency_wait();
    const int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (u < n) deg[u] = (int32_t)(row_ptr[u + 1] - row_ptr[u]);
}

__global__ void __launch_bounds__(256) k_col_deg_lower(const unsigned long long* __restrict__ keys, int64_t n_edges,
                                                      int32_t* __restrict__ col, int32_t* __restrict__ deg) {
    grid_dependency_wait();
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_edges;
         e += (int64_t)gridDim.x * blockDim.x) {
        const uint32_t v = (uint32_t)keys[e];
        col[e] = (int32_t)v;
        atomicAdd(&deg[v], 1);
    }
}

// ---- unsorted keys -> CSR without a global sort (the path of tcrnet_build / tcrnet_assemble) ----
//
// The edges of a row are few (a handful at TCR scale), so the CSR is built the way a CSR is defined.  The
// emission (or k_count_rows for caller-supplied keys) counts, for every edge (u, v), row_count[u]++ and
// deg[v]++ (fire-and-forget L2 reductions); then
//   row_ptr   = INCLUSIVE prefix sum of row_count (the end of every row)                (scan.cu)
//   k_scatter_keys   every key into a free slot of its row: bucket[--row_ptr[u]] = key; when all keys are placed
//                    row_ptr[u] has counted down to the start of row u, i.e. it is the exclusive prefix sum
//   k_rank_rows      one thread per slot: col[row_ptr[u] + #{w in row u : w < v}] = v for rows of <= kRankRow
//                    neighbours (equal keys of a caller's list: ties broken by slot); coalesced, the row is
//                    read from L1.  The thread of slot 0 adds the row length to deg[u] and queues longer rows
//   k_sort_long_rows one CTA per queued row: bitonic network in shared memory (<= kSmemRow) or in place.
// Per edge: 8 B read + 8 B written at random (scatter), 8 B read + 4 B written in order (rank), two L2
// reductions and one L2 atomic; per node 12 B + the scan.  All of it is L2-resident at TCR scale.  The result
// is the CSR a global sort of the keys yields (rows ascending by construction, neighbours by rank).
constexpr int kRankRow = 256;    // rows up to this many neighbours are ordered by ranking, one thread per edge (len^2
                                 // compares per row; measured 64 / 128 / 256 / 512 on an input with 12,715 rows of
                                 // 65..1,741 neighbours: CSR step 0.40 / 0.34 / 0.31 / 0.32 ms)
constexpr int kSmemRow = 8192;   // longer rows up to this many: bitonic network in shared memory; beyond: in place

__global__ void __launch_bounds__(256) k_count_rows(const unsigned long long* __restrict__ keys, int64_t n_keys,
                                                   int32_t* __restrict__ row_count, int32_t* __restrict__ deg) {
    grid_dependency_wait();
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_keys; e += (int64_t)gridDim.x * blockDim.x) {
        const unsigned long long k = keys[e];
        atomicAdd(&row_count[k >> 32], 1);
        atomicAdd(&deg[(uint32_t)k], 1);
    }
}

// row_ptr[u] arrives as the END of row u (inclusive prefix sum of the counts) and counts down to its start: when the
// kernel ends it IS the exclusive prefix sum.  Consecutive keys often share their row (the products of two repeated
// sequences are emitted together), so the lanes of a warp that hold the same row take their slots with ONE returning
// atomic (match.any; the returning atomics are what bounds this kernel).
//
// The number of keys is n_bound, or - a build that assembles before the host has read the edge count back - *n_dev,
// of which at most n_bound fit the buffers: beyond that nothing is written (the host will find the count too large and
// repeat the step with larger buffers).
__device__ __forceinline__ int64_t key_count(const unsigned long long* n_dev, int64_t n_bound) {
    if (!n_dev) return n_bound;
    const unsigned long long v = *n_dev;
    return v > (unsigned long long)n_bound ? -1 : (int64_t)v;  // (-1: the per-row counts describe more keys than fit)
}

__global__ void __launch_bounds__(256) k_scatter_keys(const unsigned long long* __restrict__ keys,
                                                     const unsigned long long* __restrict__ n_dev, int64_t n_bound,
                                                     unsigned long long* __restrict__ row_ptr,
                                                     unsigned long long* __restrict__ bucket) {
    grid_dependency_wait();
    const int64_t n_keys = key_count(n_dev, n_bound);
    const int lane = threadIdx.x & 31;
    const uint32_t lt_mask = (1u << lane) - 1u;
    for (int64_t e0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) & ~(int64_t)31; e0 < n_keys;
         e0 += (int64_t)gridDim.x * blockDim.x) {
        const bool valid = e0 + lane < n_keys;
        const unsigned long long k = valid ? keys[e0 + lane] : ~0ull;
        const uint32_t u = (uint32_t)(k >> 32);  // (0xffffffff is no row: n <= 2^31 - 2)
        const uint32_t same = __match_any_sync(0xffffffffu, u);
        const int leader = __ffs((int)same) - 1;
        unsigned long long end = 0;
        if (valid && lane == leader) end = atomicAdd(&row_ptr[u], (unsigned long long)(-(long long)__popc(same)));
        end = __shfl_sync(0xffffffffu, end, leader);
        if (valid) bucket[end - 1ull - (unsigned long long)__popc(same & lt_mask)] = k;
    }
}

// TIES: the keys may repeat (a caller's list); the library's own edge lists hold every pair once.
template <bool TIES>
__device__ __forceinline__ void rank_slot(const unsigned long long* __restrict__ bucket, int64_t pos,
                                          const int64_t* __restrict__ row_ptr, int32_t* __restrict__ col,
                                          int32_t* __restrict__ deg, int32_t* __restrict__ long_rows,
                                          uint32_t* __restrict__ n_long, int rank_row) {
    const unsigned long long k = bucket[pos];
    const uint32_t u = (uint32_t)(k >> 32), v = (uint32_t)k;
    const int64_t b = row_ptr[u];
    const int len = (int)(row_ptr[u + 1] - b);
    const int my = (int)(pos - b);
    if (my == 0) {
        deg[u] += len;  // the neighbours above u (those below were counted by the emission)
        if (len > rank_row) long_rows[atomicAdd(n_long, 1u)] = (int32_t)u;
    }
    if (len > rank_row) return;
    const uint32_t* a = reinterpret_cast<const uint32_t*>(bucket + b);  // the neighbour is the low word of a key
    int rank = 0;
#pragma unroll 4
    for (int i = 0; i < len; ++i) {
        const uint32_t x = __ldg(a + 2 * i);
        rank += TIES ? ((x < v) || (x == v && i < my)) : (x < v);
    }
    col[b + rank] = (int32_t)v;
}

template <bool TIES>
__global__ void __launch_bounds__(256) k_rank_rows(const unsigned long long* __restrict__ bucket,
                                                  const unsigned long long* __restrict__ n_dev, int64_t n_bound,
                                                  const int64_t* __restrict__ row_ptr, int32_t* __restrict__ col,
                                                  int32_t* __restrict__ deg, int32_t* __restrict__ long_rows,
                                                  uint32_t* __restrict__ n_long, int rank_row) {
    grid_dependency_wait();
    const int64_t n_keys = key_count(n_dev, n_bound);
    for (int64_t pos = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; pos < n_keys;
         pos += (int64_t)gridDim.x * blockDim.x)
        rank_slot<TIES>(bucket, pos, row_ptr, col, deg, long_rows, n_long, rank_row);
}


// Ascending bitonic network over the next power of two of len, the missing tail being virtual +infinity entries
// (every exchange puts the smaller value at the smaller index, so they never move).  One CTA.  The partner of element
// e at distance jj is e ^ jj, in the first stage of every k the mirror image e ^ (2 jj - 1).  Exchanges at distance
// <= 32 stay inside aligned chunks of 64 elements: a warp takes a chunk through all of them in REGISTERS (two elements
// per lane, partners by shuffle: 9 instructions per stage and lane instead of 35 through shared memory); only the
// stages of distance >= 64 go through memory, with a block barrier each.
__device__ __forceinline__ void warp_stage(int32_t& r0, int32_t& r1, int lane, int jj, bool mirror) {
    constexpr uint32_t kFull = 0xffffffffu;
    if (jj == 32) {
        if (mirror) {  // e ^ 63: the other slot of lane ^ 31
            const int32_t o0 = __shfl_xor_sync(kFull, r1, 31), o1 = __shfl_xor_sync(kFull, r0, 31);
            r0 = min(r0, o0);
            r1 = max(r1, o1);
        } else {       // e ^ 32: the other slot of this lane
            const int32_t lo = min(r0, r1);
            r1 = max(r0, r1);
            r0 = lo;
        }
    } else {
        const int m = mirror ? 2 * jj - 1 : jj;
        const int32_t o0 = __shfl_xor_sync(kFull, r0, m), o1 = __shfl_xor_sync(kFull, r1, m);
        const bool lower = (lane & jj) == 0;
        r0 = lower ? min(r0, o0) : max(r0, o0);
        r1 = lower ? min(r1, o1) : max(r1, o1);
    }
}

template <typename I>
__device__ __forceinline__ void bitonic_row(int32_t* a, I len) {
    I p2 = 64;
    while (p2 < len) p2 <<= 1;
    const I half = p2 >> 1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, n_warp = blockDim.x >> 5;
    // a chunk of 64 through the stages jj_first .. 1 of one k (k_last = 0), or through all of k = 2 .. k_last
    auto chunks = [&](int jj_first, int k_last) {
        for (I c = (I)warp * 64; c < p2; c += (I)n_warp * 64) {
            const I e0 = c + (I)lane, e1 = e0 + 32;
            int32_t r0 = e0 < len ? a[e0] : INT32_MAX, r1 = e1 < len ? a[e1] : INT32_MAX;  // (row ids are < 2^31 - 2)
            if (k_last) {
                for (int k = 2; k <= k_last; k <<= 1)
                    for (int jj = k >> 1; jj >= 1; jj >>= 1) warp_stage(r0, r1, lane, jj, jj == (k >> 1));
            } else {
                for (int jj = jj_first; jj >= 1; jj >>= 1) warp_stage(r0, r1, lane, jj, false);
            }
            if (e0 < len) a[e0] = r0;
            if (e1 < len) a[e1] = r1;
        }
        __syncthreads();
    };
    chunks(0, 64);  // sorted runs of 64
    for (I k = 128; k <= p2; k <<= 1) {
        int lg = 6;
        while (((I)2 << lg) < k) ++lg;  // jj = 1 << lg starts at k / 2
        for (I jj = k >> 1; jj >= 64; jj >>= 1, --lg) {
            const bool mirror = jj == (k >> 1);
            for (I t = threadIdx.x; t < half; t += blockDim.x) {
                const I off = t & (jj - 1);
                const I i = ((t >> lg) << (lg + 1)) + off;
                const I j = mirror ? i + 2 * (jj - off) - 1 : i + jj;
                if (j < len) {
                    const int32_t x = a[i], y = a[j];
                    if (x > y) {
                        a[i] = y;
                        a[j] = x;
                    }
                }
            }
            __syncthreads();
        }
        chunks(32, 0);
    }
}

// One CTA per queued row: ascending bitonic network over the next power of two, the missing tail being virtual
// +infinity entries (every exchange puts the smaller value at the smaller index, so they never move).
__global__ void __launch_bounds__(256) k_sort_long_rows(const int64_t* __restrict__ row_ptr,
                                                       const unsigned long long* __restrict__ bucket,
                                                       int32_t* __restrict__ col, const int32_t* __restrict__ long_rows,
                                                       const uint32_t* __restrict__ n_long) {
    grid_dependency_wait();
    __shared__ int32_t buf[kSmemRow];
    const uint32_t rows = *n_long;
    for (uint32_t r = blockIdx.x; r < rows; r += gridDim.x) {
        const int64_t u = long_rows[r];
        const int64_t b = row_ptr[u];
        const int64_t len = row_ptr[u + 1] - b;
        const bool in_smem = len <= kSmemRow;
        int32_t* a = in_smem ? buf : col + b;
        for (int64_t i = threadIdx.x; i < len; i += blockDim.x) a[i] = (int32_t)(uint32_t)bucket[b + i];
        __syncthreads();
        if (in_smem) bitonic_row<uint32_t>(a, (uint32_t)len);  // (32-bit index arithmetic: 3x fewer instructions)
        else bitonic_row<uint64_t>(a, (uint64_t)len);
        if (in_smem)
            for (int64_t i = threadIdx.x; i < len; i += blockDim.x) col[b + i] = buf[i];
        __syncthreads();
    }
}

}  // namespace

cudaError_t launch_count_rows(const unsigned long long* keys, int64_t n_keys, int32_t* row_count, int32_t* deg,
                              cudaStream_t s, int* launches) {
    if (n_keys <= 0) return cudaSuccess;
    const int64_t blocks = std::min<int64_t>((n_keys + 255) / 256, device_sm_count() * 16);
    launch_dep(k_count_rows, (unsigned)blocks, 256, 0, s, keys, n_keys, row_count, deg);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_csr_unsorted(const unsigned long long* keys, const unsigned long long* n_dev, int64_t n_bound,
                                int64_t n, int32_t* row_count, int64_t* row_ptr, unsigned long long* bucket,
                                int32_t* col, int32_t* deg, int32_t* long_rows, uint32_t* n_long, void* scan_scratch,
                                bool distinct_keys, cudaStream_t s, int* launches) {
    cudaError_t e = cudaMemsetAsync(n_long, 0, sizeof(uint32_t), s);  // (ahead of the kernels: none sits between two)
    if (e == cudaSuccess) e = inclusive_scan_i32_to_i64(row_count, row_ptr, n, scan_scratch, s, launches);
    if (e != cudaSuccess || n_bound <= 0) return e;
    // (grids: by the number of keys when the host knows it, else a fixed one - the kernels stride)
    const int64_t blocks = (n_bound + 255) / 256;
    const int64_t cap_blocks = (int64_t)device_sm_count() * (n_dev ? 16 : 32);
    launch_dep(k_scatter_keys, (unsigned)std::min<int64_t>(blocks, cap_blocks), 256, 0, s, keys, n_dev, n_bound,
               (unsigned long long*)row_ptr, bucket);
    const int rank_row = kRankRow;
    const unsigned rank_blocks = (unsigned)(n_dev ? std::min<int64_t>(blocks, (int64_t)device_sm_count() * 64) : blocks);
    if (distinct_keys) launch_dep(k_rank_rows<false>, rank_blocks, 256, 0, s, bucket, n_dev, n_bound, row_ptr, col, deg,
                                  long_rows, n_long, rank_row);
    else launch_dep(k_rank_rows<true>, rank_blocks, 256, 0, s, bucket, n_dev, n_bound, row_ptr, col, deg, long_rows,
                    n_long, rank_row);
    *launches += 2;
    return cudaGetLastError();
}

// The rows k_rank_rows queued (more than kRankRow neighbours).  Launched by the caller once it has read *n_long back
// with the build's final synchronisation and found it non-zero: repertoires without conserved ends have no such row,
// and a launch that finds nothing to do still costs 3 us.
cudaError_t launch_sort_long_rows(int64_t n, const int64_t* row_ptr, const unsigned long long* bucket, int32_t* col,
                                  const int32_t* long_rows, const uint32_t* n_long, cudaStream_t s, int* launches) {
    launch_dep(k_sort_long_rows, (unsigned)std::min<int64_t>(n, device_sm_count() * 7), 256, 0, s, row_ptr, bucket,
               col, long_rows, n_long);  // (7 CTAs of 32 KB shared memory per SM)
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_csr(const unsigned long long* sorted_keys, int64_t n_edges, int64_t n, int64_t* row_ptr,
                       int32_t* col, int32_t* deg, cudaStream_t s, int* launches) {
    launch_dep(k_row_ptr, (unsigned)((n + 1 + 255) / 256), 256, 0, s, sorted_keys, n_edges, n, row_ptr);
    launch_dep(k_deg_upper, (unsigned)((n + 255) / 256), 256, 0, s, row_ptr, n, deg);
    *launches += 2;
    if (n_edges > 0) {
        int64_t blocks = (n_edges + 255) / 256;
        if (blocks > device_sm_count() * 16) blocks = device_sm_count() * 16;
        launch_dep(k_col_deg_lower, (unsigned)blocks, 256, 0, s, sorted_keys, n_edges, col, deg);
        *launches += 1;
    }
    return cudaGetLastError();
}

}  // namespace tcrnet

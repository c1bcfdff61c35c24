// Device-wide exclusive prefix sums (row offsets, ranks of the distinct sequences, group and CSR row starts).
// Long inputs, three launches: per-tile sums -> scan of the tile sums by one CTA -> per-tile scan + offset.
// Up to kFusedTiles tiles of 1024 (every scan at TCR scale), two launches: per-tile sums -> per-tile scan, each
// CTA adding up the sums of the tiles before it itself (<= 8 loads per thread): these scans are latency-bound,
// so a launch less and four times as many CTAs matter more than the re-read sums.
// HBM-bound streaming passes: 2 reads + 1 write of the array.
#include <mutex>

#include "launch.cuh"
#include "tcrnet_internal.h"

namespace tcrnet {
namespace {

constexpr int kScanThreads = 256;
constexpr int64_t kFusedTiles = 2048;  // short path: n <= 2,097,152
__host__ __device__ constexpr int scan_items(bool fused) { return fused ? 4 : 16; }  // per thread: tiles of 1024 / 4096

template <typename T>
__device__ __forceinline__ T warp_inclusive(T v) {
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        T o = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += o;
    }
    return v;
}

// Exclusive scan of one value per thread across the CTA; *total gets the CTA sum.
template <typename T>
__device__ __forceinline__ T block_exclusive(T v, T* warp_sums /*[32]*/, T* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    T inc = warp_inclusive(v);
    if (lane == 31) warp_sums[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        T w = lane < nwarp ? warp_sums[lane] : T(0);
        T wi = warp_inclusive(w);
        warp_sums[lane] = wi - w;  // exclusive
        if (lane == 31) *total = wi;
    }
    __syncthreads();
    T r = warp_sums[warp] + inc - v;
    __syncthreads();
    return r;
}

template <typename TIn, typename TOut, bool FUSED>
__global__ void __launch_bounds__(kScanThreads) k_tile_sums(const TIn* __restrict__ in, int64_t n,
                                                           TOut* __restrict__ tile_sums) {
    grid_dependency_wait();
    constexpr int kScanItems = scan_items(FUSED), kScanTile = kScanThreads * kScanItems;
    __shared__ TOut ws[32];
    __shared__ TOut tot;
    const int64_t base = (int64_t)blockIdx.x * kScanTile;
    TOut acc = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        int64_t i = base + (int64_t)k * kScanThreads + threadIdx.x;  // coalesced
        if (i < n) acc += (TOut)in[i];
    }
    block_exclusive(acc, ws, &tot);
    if (threadIdx.x == 0) tile_sums[blockIdx.x] = tot;
}

// One CTA scans the tile sums in place (exclusive), chunk by chunk with a carry.
template <typename TOut>
__global__ void __launch_bounds__(1024) k_scan_tile_sums(TOut* __restrict__ tile_sums, int64_t n_tiles) {
    grid_dependency_wait();
    __shared__ TOut ws[32];
    __shared__ TOut tot;
    TOut carry = 0;
    for (int64_t c = 0; c < n_tiles; c += 1024) {
        int64_t i = c + threadIdx.x;
        TOut v = i < n_tiles ? tile_sums[i] : TOut(0);
        TOut ex = block_exclusive(v, ws, &tot);
        if (i < n_tiles) tile_sums[i] = carry + ex;
        carry += tot;
        __syncthreads();
    }
}

// FUSED: tile_sums holds the plain sums and this CTA adds up those of the tiles before it; else their exclusive scan.
template <typename TIn, typename TOut, bool FUSED>
__global__ void __launch_bounds__(kScanThreads) k_tile_scan(const TIn* __restrict__ in, TOut* __restrict__ out,
                                                           int64_t n, const TOut* __restrict__ tile_sums,
                                                           int write_total, int inclusive) {
    grid_dependency_wait();
    constexpr int kScanItems = scan_items(FUSED), kScanTile = kScanThreads * kScanItems;
    __shared__ TOut ws[32];
    __shared__ TOut tot;
    __shared__ TOut stage[kScanTile];
    const int64_t base = (int64_t)blockIdx.x * kScanTile;
    TOut tile_base;
    if (FUSED) {
        TOut before = 0;
        for (unsigned t = threadIdx.x; t < blockIdx.x; t += kScanThreads) before += tile_sums[t];
        block_exclusive(before, ws, &tot);
        tile_base = tot;
        __syncthreads();  // tot is reused below
    } else {
        tile_base = tile_sums[blockIdx.x];
    }
    // coalesced load into shared memory, then each thread owns kScanItems consecutive items
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        int idx = k * kScanThreads + threadIdx.x;
        int64_t i = base + idx;
        stage[idx] = i < n ? (TOut)in[i] : TOut(0);
    }
    __syncthreads();
    TOut local[kScanItems];
    TOut acc = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        local[k] = acc;
        acc += stage[threadIdx.x * kScanItems + k];
    }
    TOut ex = block_exclusive(acc, ws, &tot) + tile_base;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) stage[threadIdx.x * kScanItems + k] = local[k] + ex;
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        int idx = k * kScanThreads + threadIdx.x;
        int64_t i = base + idx;
        if (i < n) out[i] = stage[idx] + (inclusive ? (TOut)in[i] : TOut(0));
    }
    if (write_total && blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) out[n] = tile_base + tot;
}

template <typename TIn, typename TOut>
cudaError_t scan_impl(const TIn* in, TOut* out, int64_t n, bool write_total, void* scratch, cudaStream_t s,
                      int* launches, bool inclusive = false) {
    if (n <= 0) {
        if (write_total) return cudaMemsetAsync(out, 0, sizeof(TOut), s);
        return cudaSuccess;
    }
    TOut* sums = static_cast<TOut*>(scratch);
    const int64_t small_tile = kScanThreads * scan_items(true), big_tile = kScanThreads * scan_items(false);
    if ((n + small_tile - 1) / small_tile <= kFusedTiles) {
        const int64_t tiles = (n + small_tile - 1) / small_tile;
        launch_dep(k_tile_sums<TIn, TOut, true>, (unsigned)tiles, kScanThreads, 0, s, in, n, sums);
        launch_dep(k_tile_scan<TIn, TOut, true>, (unsigned)tiles, kScanThreads, 0, s, in, out, n, sums,
                   write_total ? 1 : 0, inclusive ? 1 : 0);
        *launches += 2;
        return cudaGetLastError();
    }
    const int64_t tiles = (n + big_tile - 1) / big_tile;
    launch_dep(k_tile_sums<TIn, TOut, false>, (unsigned)tiles, kScanThreads, 0, s, in, n, sums);
    launch_dep(k_scan_tile_sums<TOut>, 1, 1024, 0, s, sums, tiles);
    launch_dep(k_tile_scan<TIn, TOut, false>, (unsigned)tiles, kScanThreads, 0, s, in, out, n, sums,
               write_total ? 1 : 0, inclusive ? 1 : 0);
    *launches += 3;
    return cudaGetLastError();
}

}  // namespace

size_t scan_scratch_bytes(int64_t n) {
    const int64_t tile = kScanThreads * scan_items(true);  // the smaller tile: an upper bound for both paths
    const int64_t tiles = (n + tile - 1) / tile;
    return (size_t)(tiles > 0 ? tiles : 1) * sizeof(int64_t);
}

cudaError_t exclusive_scan_i32_to_i64(const int32_t* in, int64_t* out, int64_t n, bool write_total, void* scratch,
                                      cudaStream_t s, int* launches) {
    return scan_impl<int32_t, int64_t>(in, out, n, write_total, scratch, s, launches);
}

// out[i] = in[0] + ... + in[i]; out[n] = the total
cudaError_t inclusive_scan_i32_to_i64(const int32_t* in, int64_t* out, int64_t n, void* scratch, cudaStream_t s,
                                      int* launches) {
    return scan_impl<int32_t, int64_t>(in, out, n, true, scratch, s, launches, true);
}

cudaError_t exclusive_scan_u32_total(const uint32_t* in, uint32_t* out, int64_t n, void* scratch, cudaStream_t s,
                                     int* launches) {
    return scan_impl<uint32_t, uint32_t>(in, out, n, true, scratch, s, launches);
}

}  // namespace tcrnet

// ---- tcrnet_row_ptr_noalloc (tcrnet.h): the prefix sum with its scratch in a static device array ----
// For callers that cannot call cudaMalloc (CUDA graph capture, serving loops, harnesses that forbid it): the same two
// kernels as exclusive_scan_i32_to_i64, their per-tile sums in a file-scope array instead of a buffer of the context.
// Every GPU that loads the library holds the array (16 KB) until exit.
namespace {

constexpr int64_t kNoAllocTiles = tcrnet::kFusedTiles;  // tiles of 1024 counts: TCRNET_NOALLOC_MAX_ROWS counts
static_assert(kNoAllocTiles * tcrnet::kScanThreads * tcrnet::scan_items(true) == TCRNET_NOALLOC_MAX_ROWS,
              "the header states the limit");
static __device__ __align__(256) unsigned long long g_noalloc_tile_sums[kNoAllocTiles];

// In host code the array's name is a host-side stand-in, not a device address: the kernels get what
// cudaGetSymbolAddress returns on the device that is current, looked up once per device.
constexpr int kMaxDevices = 64;
void* g_noalloc_addr[kMaxDevices];
bool g_noalloc_have[kMaxDevices];
std::mutex g_noalloc_mutex;

cudaError_t noalloc_scratch(void** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_have[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_tile_sums);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_noalloc_addr[dev] = p;
        g_noalloc_have[dev] = true;
    }
    *out = g_noalloc_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int tcrnet_row_ptr_noalloc(const int32_t* counts_dev, int64_t n, int64_t* row_ptr_dev, void* cuda_stream,
                                      int* cuda_error_out) {
    if (cuda_error_out) *cuda_error_out = 0;
    if (n < 0 || !row_ptr_dev || (n > 0 && !counts_dev)) return TCRNET_ERR_ARG;
    if (n > TCRNET_NOALLOC_MAX_ROWS) return TCRNET_ERR_CAPACITY;  // (before anything is read or launched)
    void* scratch = nullptr;
    cudaError_t e = noalloc_scratch(&scratch);
    int launches = 0;
    // (the sums of the tiles in use are written by the first kernel before the second reads them: nothing in the
    // array has to start at zero, whatever the last call left there)
    if (e == cudaSuccess)
        e = tcrnet::scan_impl<int32_t, int64_t>(counts_dev, row_ptr_dev, n, true, scratch, (cudaStream_t)cuda_stream,
                                                &launches);
    if (e != cudaSuccess) {
        if (cuda_error_out) *cuda_error_out = (int)e;
        (void)cudaGetLastError();
        return TCRNET_ERR_CUDA;
    }
    return TCRNET_OK;
}

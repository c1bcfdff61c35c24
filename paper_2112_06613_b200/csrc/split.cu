// One stable counting-sort pass over an 8-bit digit (the building block of the length sort in
// step A1 and of the LSD radix sort of the edge keys in step A6).
//
//   hist    : per-CTA digit counts, stored digit-major (hist[d * blocks + b]) so that ONE
//             exclusive scan over the flat array yields, for every (digit, CTA), the first
//             output slot of that CTA's items with that digit.
//   scatter : each CTA re-reads its items in order and ranks equal digits by position
//             (warp: __match_any_sync + popc of the lower lanes; CTA: per-warp counts in
//             shared memory), so the pass is stable.
#include "tcrnet_internal.h"

namespace tcrnet {
namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kRounds = 16;
constexpr int kItemsPerBlock = kThreads * kRounds;  // 4096

struct LengthDigit {
    const int32_t* lengths;
    __device__ __forceinline__ uint32_t digit(int64_t i) const {
        int32_t l = lengths[i];
        return (l < 0 || l > kMaxLen) ? 0u : (uint32_t)l;  // invalid lengths are reported elsewhere
    }
};

struct KeyDigit {
    const unsigned long long* keys;
    int shift;
    __device__ __forceinline__ uint32_t digit(int64_t i) const { return (uint32_t)(keys[i] >> shift) & 255u; }
};

template <typename D>
__global__ void __launch_bounds__(kThreads) k_split_hist(D src, int64_t n, uint32_t* __restrict__ hist,
                                                        uint32_t blocks) {
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * kItemsPerBlock;
#pragma unroll 4
    for (int r = 0; r < kRounds; ++r) {
        int64_t i = base + (int64_t)r * kThreads + threadIdx.x;
        if (i < n) atomicAdd(&h[src.digit(i)], 1u);
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * blocks + blockIdx.x] = h[threadIdx.x];
}

struct PermSink {
    int32_t* perm;
    __device__ __forceinline__ void put(int64_t pos, int64_t i) const { perm[pos] = (int32_t)i; }
};

struct KeySink {
    const unsigned long long* in;
    unsigned long long* out;
    __device__ __forceinline__ void put(int64_t pos, int64_t i) const { out[pos] = in[i]; }
};

template <typename D, typename S>
__global__ void __launch_bounds__(kThreads) k_split_scatter(D src, S sink, int64_t n,
                                                           const uint32_t* __restrict__ hist_scanned,
                                                           uint32_t blocks) {
    __shared__ uint32_t base[256];
    __shared__ uint32_t wcount[kWarps][256];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    base[threadIdx.x] = hist_scanned[(size_t)threadIdx.x * blocks + blockIdx.x];
#pragma unroll
    for (int w = 0; w < kWarps; ++w) wcount[w][threadIdx.x] = 0;
    __syncthreads();
    const int64_t first = (int64_t)blockIdx.x * kItemsPerBlock;
    for (int r = 0; r < kRounds; ++r) {
        const int64_t i = first + (int64_t)r * kThreads + threadIdx.x;
        if (first + (int64_t)r * kThreads >= n) break;  // CTA-uniform
        const bool valid = i < n;
        const uint32_t d = valid ? src.digit(i) : (256u + lane);  // invalid lanes match nobody
        const uint32_t peers = __match_any_sync(0xffffffffu, d);
        const uint32_t rank = __popc(peers & ((1u << lane) - 1u));
        if (valid && rank == 0) wcount[warp][d] = __popc(peers);
        __syncthreads();
        if (valid) {
            uint32_t off = base[d];
            for (int w = 0; w < warp; ++w) off += wcount[w][d];
            sink.put((int64_t)off + rank, i);
        }
        __syncthreads();
        uint32_t add = 0;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) {
            add += wcount[w][threadIdx.x];
            wcount[w][threadIdx.x] = 0;
        }
        base[threadIdx.x] += add;
        __syncthreads();
    }
}

template <typename D, typename S>
cudaError_t split_impl(D src, S sink, int64_t n, uint32_t* hist, uint32_t* hist_scanned, void* scan_scratch,
                       cudaStream_t s, int* launches) {
    if (n <= 0) return cudaSuccess;
    const int64_t blocks = split_num_blocks(n);
    k_split_hist<D><<<(unsigned)blocks, kThreads, 0, s>>>(src, n, hist, (uint32_t)blocks);
    *launches += 1;
    cudaError_t e = exclusive_scan_u32(hist, hist_scanned, 256 * blocks, scan_scratch, s, launches);
    if (e != cudaSuccess) return e;
    k_split_scatter<D, S><<<(unsigned)blocks, kThreads, 0, s>>>(src, sink, n, hist_scanned, (uint32_t)blocks);
    *launches += 1;
    return cudaGetLastError();
}

}  // namespace

int64_t split_num_blocks(int64_t n) { return n > 0 ? (n + kItemsPerBlock - 1) / kItemsPerBlock : 1; }

cudaError_t split_by_length(const int32_t* lengths, int64_t n, int32_t* perm_out, uint32_t* hist,
                            uint32_t* hist_scanned, void* scan_scratch, cudaStream_t s, int* launches) {
    return split_impl(LengthDigit{lengths}, PermSink{perm_out}, n, hist, hist_scanned, scan_scratch, s, launches);
}

cudaError_t split_keys_u64(const unsigned long long* in, unsigned long long* out, int64_t n, int shift,
                           uint32_t* hist, uint32_t* hist_scanned, void* scan_scratch, cudaStream_t s,
                           int* launches) {
    return split_impl(KeyDigit{in, shift}, KeySink{in, out}, n, hist, hist_scanned, scan_scratch, s, launches);
}

}  // namespace tcrnet

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

// Digits of the sequence sort (step A1).  `perm_in` is the current order (NULL = identity).
struct LengthDigit {
    const int32_t* lengths;
    const int32_t* perm_in;
    __device__ __forceinline__ uint32_t digit(int64_t i) const {
        const int32_t l = lengths[perm_in ? perm_in[i] : i];
        return (l < 0 || l > kMaxLen) ? 0u : (uint32_t)l;  // invalid lengths are reported elsewhere
    }
};

struct ResidueDigit {  // residue at position k (0 = past the end), for the lexicographic sub-order
    const uint8_t* residues;
    const int64_t* offsets;
    const int32_t* lengths;
    const int32_t* perm_in;
    int k;
    __device__ __forceinline__ uint32_t digit(int64_t i) const {
        const int64_t o = perm_in ? perm_in[i] : i;
        const int32_t l = lengths[o];
        if (l < 1 || l > kMaxLen || k >= l) return 0u;
        const uint32_t c = (uint32_t)residues[offsets[o] + k] - (uint32_t)'A';
        return (c < 26u ? c : 26u) + 1u;  // invalid residues are reported by the pack kernel
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
    const int32_t* perm_in;
    int32_t* perm_out;
    __device__ __forceinline__ void put(int64_t pos, int64_t i) const {
        perm_out[pos] = perm_in ? perm_in[i] : (int32_t)i;
    }
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

cudaError_t split_by_length(const int32_t* lengths, const int32_t* perm_in, int64_t n, int32_t* perm_out,
                            uint32_t* hist, uint32_t* hist_scanned, void* scan_scratch, cudaStream_t s,
                            int* launches) {
    return split_impl(LengthDigit{lengths, perm_in}, PermSink{perm_in, perm_out}, n, hist, hist_scanned,
                      scan_scratch, s, launches);
}

cudaError_t split_by_residue(const uint8_t* residues, const int64_t* offsets, const int32_t* lengths,
                             const int32_t* perm_in, int k, int64_t n, int32_t* perm_out, uint32_t* hist,
                             uint32_t* hist_scanned, void* scan_scratch, cudaStream_t s, int* launches) {
    return split_impl(ResidueDigit{residues, offsets, lengths, perm_in, k}, PermSink{perm_in, perm_out}, n, hist,
                      hist_scanned, scan_scratch, s, launches);
}

cudaError_t split_keys_u64(const unsigned long long* in, unsigned long long* out, int64_t n, int shift,
                           uint32_t* hist, uint32_t* hist_scanned, void* scan_scratch, cudaStream_t s,
                           int* launches) {
    return split_impl(KeyDigit{in, shift}, KeySink{in, out}, n, hist, hist_scanned, scan_scratch, s, launches);
}

}  // namespace tcrnet

// Stable LSD radix sort over kRadixBits-bit (9) digits of 64-bit keys, with an optional 32-bit payload: the sequence
// sort of step A1 (composite (length, first residues) keys, payload = caller's row).  HBM/L2-bound
// streaming; three launches per pass, no spinning on other CTAs:
//
//   k_radix_hist     per tile of 4096 (1024 for short inputs) keys, the 512 digit counts (shared-memory atomics), stored digit-major
//                    (hist[d * tiles + tile]) and added to the pass's global digit totals;
//   k_radix_scan     CTA d turns row d of `hist` into global output positions: the total of all smaller
//                    digits (from the global totals) + the exclusive prefix over the tiles;
//   k_radix_scatter  each warp owns 512 (128) consecutive keys of its tile and ranks equal digits in order
//                    (__match_any_sync + a warp-private running count in shared memory, no CTA barrier
//                    inside the loop), the 8 warp counts are chained once, keys go straight to their
//                    final slot.  Order inside a digit = input order, so every pass is stable.
#include <utility>

#include "launch.cuh"
#include "tcrnet_internal.h"

namespace tcrnet {
namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr uint32_t kFull = 0xffffffffu;
constexpr int kDigits = 1 << kRadixBits;  // 512: the 36-bit sequence key takes 4 passes
static_assert(kDigits % kThreads == 0 && kDigits <= 0x8000, "digit loops stride by the CTA; rank | digit << 16");
// keys per thread (ROUNDS): 16 for long inputs (4096 keys per CTA, 512 consecutive keys per warp); 4 below
// kSmallN keys, where 4096-key tiles would leave most SMs without a CTA and every pass is latency-bound
constexpr int64_t kSmallN = (int64_t)1 << 22;
__host__ __device__ constexpr int rounds_for(int64_t n) { return n < kSmallN ? 4 : 16; }

template <int kRounds>
__global__ void __launch_bounds__(kThreads) k_radix_hist(const unsigned long long* __restrict__ keys, int64_t n,
                                                        int shift, uint32_t* __restrict__ hist,
                                                        uint32_t* __restrict__ totals, uint32_t tiles) {
    grid_dependency_wait();
    constexpr int kTile = kThreads * kRounds;
    __shared__ uint32_t h[kDigits];
    for (int d = threadIdx.x; d < kDigits; d += kThreads) h[d] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * kTile;
#pragma unroll 4
    for (int r = 0; r < kRounds; ++r) {
        const int64_t i = base + (int64_t)r * kThreads + threadIdx.x;
        if (i < n) atomicAdd(&h[(uint32_t)(keys[i] >> shift) & (uint32_t)(kDigits - 1)], 1u);
    }
    __syncthreads();
    for (int d = threadIdx.x; d < kDigits; d += kThreads) {
        const uint32_t c = h[d];
        hist[(size_t)d * tiles + blockIdx.x] = c;
        if (c) atomicAdd(&totals[d], c);
    }
}

// Row d of hist (tiles entries) -> first output slot of (digit d, tile t), in place.
__global__ void __launch_bounds__(kThreads) k_radix_scan(uint32_t* __restrict__ hist,
                                                        const uint32_t* __restrict__ totals, uint32_t tiles) {
    grid_dependency_wait();
    __shared__ uint32_t wsum[kWarps];
    const uint32_t d = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // total of the smaller digits
    uint32_t below = 0u;
    for (uint32_t t = tid; t < d; t += kThreads) below += totals[t];
    below = __reduce_add_sync(kFull, below);
    if (lane == 0) wsum[warp] = below;
    __syncthreads();
    uint32_t digit_base = 0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) digit_base += wsum[w];
    __syncthreads();
    // each thread owns a contiguous chunk of the row
    uint32_t* row = hist + (size_t)d * tiles;
    const uint32_t per = (tiles + kThreads - 1) / kThreads;
    const uint32_t b = min(tid * per, tiles), e = min(b + per, tiles);
    uint32_t sum = 0;
    for (uint32_t t = b; t < e; ++t) sum += row[t];
    // exclusive scan of the 256 partial sums (warp scan + warp totals)
    uint32_t incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(kFull, incl, o);
        if ((int)lane >= o) incl += v;
    }
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    uint32_t run = digit_base + incl - sum;
    for (uint32_t w = 0; w < warp; ++w) run += wsum[w];
    for (uint32_t t = b; t < e; ++t) {
        const uint32_t c = row[t];
        row[t] = run;
        run += c;
    }
}

template <bool HAS_VAL, int kRounds>
__global__ void __launch_bounds__(kThreads) k_radix_scatter(const unsigned long long* __restrict__ keys_in,
                                                           unsigned long long* __restrict__ keys_out,
                                                           const int32_t* __restrict__ vals_in,
                                                           int32_t* __restrict__ vals_out, int64_t n, int shift,
                                                           const uint32_t* __restrict__ scanned, uint32_t tiles) {
    grid_dependency_wait();
    constexpr int kTile = kThreads * kRounds, kWarpItems = 32 * kRounds;
    __shared__ uint32_t wh[kWarps][kDigits];  // per warp: running digit counts, then first output slots
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int d = tid; d < kDigits; d += kThreads) {
#pragma unroll
        for (int w = 0; w < kWarps; ++w) wh[w][d] = 0;
    }
    __syncthreads();
    const int64_t first = (int64_t)blockIdx.x * kTile + (int64_t)warp * kWarpItems + lane;
    const uint32_t lt = (1u << lane) - 1u;
    unsigned long long key[kRounds];
    uint32_t rank[kRounds];  // rank among the warp's keys of the same digit | digit << 16 (0xffffffff: no key)
#pragma unroll
    for (int r = 0; r < kRounds; ++r) {
        const int64_t i = first + r * 32;
        const bool valid = i < n;
        key[r] = valid ? keys_in[i] : 0ull;
        // (invalid lanes match nobody)
        const uint32_t d = valid ? (uint32_t)(key[r] >> shift) & (uint32_t)(kDigits - 1) : kDigits + lane;
        const uint32_t peers = __match_any_sync(kFull, d);
        const int leader = __ffs((int)peers) - 1;
        uint32_t old = 0;
        if (valid && (int)lane == leader) {
            old = wh[warp][d];
            wh[warp][d] = old + __popc(peers);
        }
        old = __shfl_sync(kFull, old, leader);
        rank[r] = valid ? (old + __popc(peers & lt)) | (d << 16) : 0xffffffffu;
        __syncwarp();
    }
    __syncthreads();
    for (int d = tid; d < kDigits; d += kThreads) {
        uint32_t run = scanned[(size_t)d * tiles + blockIdx.x];
#pragma unroll
        for (int w = 0; w < kWarps; ++w) {
            const uint32_t c = wh[w][d];
            wh[w][d] = run;
            run += c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kRounds; ++r) {
        if (rank[r] != 0xffffffffu) {
            const uint32_t pos = wh[warp][rank[r] >> 16] + (rank[r] & 0xffffu);
            keys_out[pos] = key[r];
            if (HAS_VAL) vals_out[pos] = vals_in[first + r * 32];
        }
    }
}

}  // namespace

int64_t radix_tiles(int64_t n) {
    const int64_t tile = (int64_t)kThreads * rounds_for(n);
    return n > 0 ? (n + tile - 1) / tile : 1;
}

size_t radix_scratch_bytes(int64_t n) {
    return ((size_t)radix_tiles(n) * kDigits + (size_t)kRadixMaxPasses * kDigits) * sizeof(uint32_t);
}

cudaError_t radix_clear_totals(void* scratch, cudaStream_t s) {
    return cudaMemsetAsync(scratch, 0, sizeof(uint32_t) * kRadixMaxPasses * kDigits, s);
}

cudaError_t radix_sort_u64(unsigned long long* keys_a, unsigned long long* keys_b, int32_t* vals_a, int32_t* vals_b,
                           int64_t n, const int* shifts, int n_passes, void* scratch, cudaStream_t s, int* launches,
                           bool* result_in_b, bool totals_cleared) {
    *result_in_b = false;
    if (n <= 1 || n_passes <= 0) return cudaSuccess;
    if (n_passes > kRadixMaxPasses || n > 0x7fffffffLL) return cudaErrorInvalidValue;
    const uint32_t tiles = (uint32_t)radix_tiles(n);
    uint32_t* totals = (uint32_t*)scratch;                     // [kRadixMaxPasses][kDigits]
    uint32_t* hist = totals + kRadixMaxPasses * kDigits;       // [kDigits][tiles]
    cudaError_t e = totals_cleared ? cudaSuccess : radix_clear_totals(scratch, s);
    if (e != cudaSuccess) return e;
    const bool has_val = vals_a != nullptr;
    const bool small = rounds_for(n) == 4;
    for (int p = 0; p < n_passes; ++p) {
        if (small) launch_dep(k_radix_hist<4>, tiles, kThreads, 0, s, keys_a, n, shifts[p], hist,
                              totals + p * kDigits, tiles);
        else launch_dep(k_radix_hist<16>, tiles, kThreads, 0, s, keys_a, n, shifts[p], hist, totals + p * kDigits,
                        tiles);
        launch_dep(k_radix_scan, kDigits, kThreads, 0, s, hist, totals + p * kDigits, tiles);
        if (has_val && small)
            launch_dep(k_radix_scatter<true, 4>, tiles, kThreads, 0, s, keys_a, keys_b, vals_a, vals_b, n, shifts[p],
                       hist, tiles);
        else if (has_val)
            launch_dep(k_radix_scatter<true, 16>, tiles, kThreads, 0, s, keys_a, keys_b, vals_a, vals_b, n, shifts[p],
                       hist, tiles);
        else if (small)
            launch_dep(k_radix_scatter<false, 4>, tiles, kThreads, 0, s, keys_a, keys_b, nullptr, nullptr, n,
                       shifts[p], hist, tiles);
        else
            launch_dep(k_radix_scatter<false, 16>, tiles, kThreads, 0, s, keys_a, keys_b, nullptr, nullptr, n,
                       shifts[p], hist, tiles);
        *launches += 3;
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        std::swap(keys_a, keys_b);
        std::swap(vals_a, vals_b);
        *result_in_b = !*result_in_b;
    }
    return cudaSuccess;
}

}  // namespace tcrnet

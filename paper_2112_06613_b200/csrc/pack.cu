// Step A1 (pack): validation, length histogram and the re-layout of the sequences into the
// tables the distance kernels read (residues "saved as a number ... BYTE";
// north_star subsystem (1): 5-bit residue codes, sorted by length, bucketed by length).
//
//   pat : one row per sorted position, one residue code (0..25) per byte, row stride
//         pat_stride bytes (multiple of 16), padded with 0xff - read once per work item to
//         build the Peq match masks.  Written on demand, like txt.
//   txt : per length bucket, one row of round_up(len,4) 32-bit words per sequence holding the
//         residue code of each column, padded with kPadCode - streamed into shared memory
//         and read with one broadcast 128-bit load per four columns.  The code sits in a
//         32-bit word so that the per-column Peq address is a single IMAD (code * row_bytes
//         + lane offset) on the FMA pipe, leaving the ALU pipe to the bit-vector recurrence.
//         Written on demand (k_rows_from_planes): only the prefix-trie / text-chunk kernels read it.
//   planes : one row of 8 words per sorted position: plane k = bit k of the 5-bit code of every residue
//         (north_star (1): 5-bit codes, here one bit of the code per word so that a residue-wise comparison of two
//         sequences under any shift is five XORs) + the length - what the segment join reads (segjoin.cu).
#include <algorithm>

#include "launch.cuh"
#include "tcrnet_internal.h"

namespace tcrnet {
namespace {

// n_dev != NULL: the number of rows is read from device memory (it is at most n)
__global__ void __launch_bounds__(256) k_length_hist(const int32_t* __restrict__ lengths, int64_t n,
                                                    const uint32_t* __restrict__ n_dev,
                                                    unsigned long long* __restrict__ hist,
                                                    uint32_t* __restrict__ flags) {
    grid_dependency_wait();
    __shared__ uint32_t h[kNumLen];
    if (n_dev) n = min(n, (int64_t)*n_dev);
    for (int i = threadIdx.x; i < kNumLen; i += blockDim.x) h[i] = 0;
    __syncthreads();
    bool bad = false;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        int32_t l = lengths[i];
        if (l < 1 || l > kMaxLen) {
            bad = true;
            l = 0;  // same clamp as the length sort
        }
        atomicAdd(&h[l], 1u);
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(flags, kFlagBadLength);
    for (int i = threadIdx.x; i < kNumLen; i += blockDim.x)
        if (h[i]) atomicAdd(&hist[i], (unsigned long long)h[i]);
}

// Sort key of the sequence sort: (length - 1 in 6 bits, first kSortPrefix residues as 5-bit digits, 0 = past the
// end, 27 = not a letter); the payload of row i is i.  Invalid lengths / residues are reported by
// k_length_hist / k_pack, here they only have to land somewhere.
__global__ void __launch_bounds__(256) k_seq_keys(const uint8_t* __restrict__ residues,
                                                 const int64_t* __restrict__ offsets,
                                                 const int32_t* __restrict__ lengths, int64_t n,
                                                 unsigned long long* __restrict__ keys, int32_t* __restrict__ vals) {
    grid_dependency_wait();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int32_t l = lengths[i];
    if (l < 1 || l > kMaxLen) l = 0;  // (the load fails on such a row; it only has to land somewhere)
    const uint8_t* src = residues + offsets[i];
    unsigned long long key = (unsigned long long)(uint32_t)(l > 0 ? l - 1 : 0);
#pragma unroll
    for (int k = 0; k < kSortPrefix; ++k) {
        uint32_t d = 0u;
        if (k < l) {
            const uint32_t c = (uint32_t)src[k] - (uint32_t)'A';
            d = (c < 26u ? c : 26u) + 1u;
        }
        key = (key << 5) | d;
    }
    keys[i] = key;
    vals[i] = (int32_t)i;
}

// One thread per sorted position: the residues of the row become its bit-plane row (8 words of W: planes 0..4, the
// length, two zero words).  A collapsed load (dedup.cu) arrives with perm[s] = uid of the distinct sequence; perm[s] is
// re-coded on the way out: the row itself for a sequence that one row has, kGroupFlag | uid for a shared one.
// Every sample_stride-th CTA also counts which residue stands at each of the first / last kPosStat positions of its
// sequences (pos_hist[0][p][c]: residue c at position p; [1][p][c]: at position len - 1 - p): the segment join cuts
// the texts where that makes its segments equally informative (tcrnet_api.cu: make_join_tables).  A sample is enough -
// any cut is exact, the statistics only shorten the candidate lists.
template <typename W>
__global__ void __launch_bounds__(256) k_pack(const uint8_t* __restrict__ residues,
                                             const int64_t* __restrict__ offsets,
                                             const int32_t* __restrict__ lengths,
                                             int32_t* __restrict__ perm, int64_t n,
                                             W* __restrict__ planes, uint32_t* __restrict__ flags,
                                             const uint32_t* __restrict__ group_start,
                                             const int32_t* __restrict__ members, uint32_t* __restrict__ pos_hist,
                                             uint32_t sample_stride) {
    grid_dependency_wait();
    __shared__ uint32_t ph[2 * kPosStat * 32];
    const bool sampled = pos_hist != nullptr && blockIdx.x % sample_stride == 0;
    if (sampled) {
        for (int i = threadIdx.x; i < 2 * kPosStat * 32; i += blockDim.x) ph[i] = 0u;
        __syncthreads();
    }
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;  // sorted position
    bool bad = false;
    if (s < n) {
        const int32_t o = perm[s];
        const int32_t len = lengths[o];
        const uint8_t* src = residues + offsets[o];
        W pl[5] = {W(0), W(0), W(0), W(0), W(0)};
        for (int i = 0; i < len; ++i) {
            uint32_t c = (uint32_t)src[i] - (uint32_t)'A';
            if (c >= (uint32_t)kNumCodes) {
                bad = true;
                c = 0;
            }
#pragma unroll
            for (int b = 0; b < 5; ++b) pl[b] |= (W)((c >> b) & 1u) << i;
        }
        // (a loop of its own: inside the loop above it doubled the kernel's duration for every CTA; every 8th row only:
        // hot residues serialise the shared-memory atomics)
        if (sampled && (threadIdx.x & 7) == 0 && !bad)
            for (int i = 0; i < len; ++i) {
                const uint32_t c = (uint32_t)src[i] - (uint32_t)'A';
                if (i < kPosStat) atomicAdd(&ph[i * 32 + c], 1u);
                if (len - 1 - i < kPosStat) atomicAdd(&ph[(kPosStat + len - 1 - i) * 32 + c], 1u);
            }
        W* row = planes + (size_t)s * kPlaneWords;
        if (sizeof(W) == 4) {
            uint4* r4 = reinterpret_cast<uint4*>(row);
            r4[0] = make_uint4((uint32_t)pl[0], (uint32_t)pl[1], (uint32_t)pl[2], (uint32_t)pl[3]);
            r4[1] = make_uint4((uint32_t)pl[4], (uint32_t)len, 0u, 0u);
        } else {
            ulonglong2* r2 = reinterpret_cast<ulonglong2*>(row);
            r2[0] = make_ulonglong2((unsigned long long)pl[0], (unsigned long long)pl[1]);
            r2[1] = make_ulonglong2((unsigned long long)pl[2], (unsigned long long)pl[3]);
            r2[2] = make_ulonglong2((unsigned long long)pl[4], (unsigned long long)len);
            r2[3] = make_ulonglong2(0ull, 0ull);
        }
        if (group_start) {
            const uint32_t b = group_start[o];
            perm[s] = group_start[o + 1] - b == 1u ? members[b] : (int32_t)(kGroupFlag | (uint32_t)o);
        }
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(flags, kFlagBadResidue);
    if (sampled)  // (the barrier above has made the counts of the CTA visible)
        for (int i = threadIdx.x; i < 2 * kPosStat * 32; i += blockDim.x)
            if (ph[i]) atomicAdd(pos_hist + i, ph[i]);
}

// The rows of the prefix-trie / text-chunk kernels from the bit-plane rows, written only when a build needs those
// kernels (tcrnet_api.cu: ensure_text_tables): pat = one residue code per byte, 0xff beyond the sequence, 128-bit
// stores; txt = one 32-bit word per column, padded with kPadCode, one 128-bit store per four columns.
template <typename W>
__global__ void __launch_bounds__(256) k_rows_from_planes(const W* __restrict__ planes, int64_t n,
                                                         const __grid_constant__ LengthTable lt, int pat_stride,
                                                         uint8_t* __restrict__ pat, uint32_t* __restrict__ txt) {
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const W* row = planes + (size_t)s * kPlaneWords;
    W pl[5];
#pragma unroll
    for (int b = 0; b < 5; ++b) pl[b] = row[b];
    const int len = (int)row[5];
    uint4* prow = reinterpret_cast<uint4*>(pat + (size_t)s * pat_stride);
    const int rw = lt.row_words[len];
    uint4* trow = reinterpret_cast<uint4*>(txt + lt.txt_base[len] + (int64_t)(s - lt.start[len]) * rw);
    for (int i0 = 0; i0 < pat_stride; i0 += 16) {
        uint32_t c[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const int i = i0 + k;
            c[k] = 0xffu;
            if (i < len) {
                c[k] = 0u;
#pragma unroll
                for (int b = 0; b < 5; ++b) c[k] |= (uint32_t)((pl[b] >> i) & W(1)) << b;
            }
        }
        uint32_t w4[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) w4[k] = c[4 * k] | (c[4 * k + 1] << 8) | (c[4 * k + 2] << 16) | (c[4 * k + 3] << 24);
        prow[i0 >> 4] = make_uint4(w4[0], w4[1], w4[2], w4[3]);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int i = i0 + 4 * k;  // text columns i .. i+3
            if (i < rw) {
                uint32_t t[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) t[q] = i + q < len ? c[4 * k + q] : (uint32_t)kPadCode;
                trow[i >> 2] = make_uint4(t[0], t[1], t[2], t[3]);
            }
        }
    }
}

}  // namespace

int device_sm_count() {
    static int cached[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    if (cached[dev] == 0) {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) {
            (void)cudaGetLastError();
            return 148;
        }
        cached[dev] = v;
    }
    return cached[dev];
}

cudaError_t launch_length_hist(const int32_t* lengths, int64_t n, const uint32_t* n_dev, unsigned long long* hist,
                               uint32_t* flags, cudaStream_t s, int* launches) {
    int64_t blocks = (n + 255) / 256;
    if (blocks > device_sm_count() * 8) blocks = device_sm_count() * 8;
    launch_dep(k_length_hist, (unsigned)blocks, 256, 0, s, lengths, n, n_dev, hist, flags);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_seq_keys(const uint8_t* residues, const int64_t* offsets, const int32_t* lengths, int64_t n,
                            unsigned long long* keys, int32_t* vals, cudaStream_t s, int* launches) {
    if (n <= 0) return cudaSuccess;
    launch_dep(k_seq_keys, (unsigned)((n + 255) / 256), 256, 0, s, residues, offsets, lengths, n, keys, vals);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_pack(const uint8_t* residues, const int64_t* offsets, const int32_t* lengths, int32_t* perm, int64_t n,
                        void* planes, bool wide_planes, uint32_t* flags, const uint32_t* group_start,
                        const int32_t* members, uint32_t* pos_hist, cudaStream_t s, int* launches) {
    const unsigned blocks = (unsigned)((n + 255) / 256);
    const uint32_t stride = std::max(1u, blocks / 128u);  // about 128 CTAs x 32 rows = 4,096 sequences are sampled
    if (wide_planes)
        launch_dep(k_pack<uint64_t>, blocks, 256, 0, s, residues, offsets, lengths, perm, n, (uint64_t*)planes, flags,
                   group_start, members, pos_hist, stride);
    else
        launch_dep(k_pack<uint32_t>, blocks, 256, 0, s, residues, offsets, lengths, perm, n, (uint32_t*)planes, flags,
                   group_start, members, pos_hist, stride);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_rows_from_planes(const void* planes, bool wide_planes, int64_t n, const LengthTable& lt, int pat_stride,
                                    uint8_t* pat, uint32_t* txt, cudaStream_t s, int* launches) {
    if (n <= 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    if (wide_planes) k_rows_from_planes<uint64_t><<<blocks, 256, 0, s>>>((const uint64_t*)planes, n, lt, pat_stride, pat, txt);
    else k_rows_from_planes<uint32_t><<<blocks, 256, 0, s>>>((const uint32_t*)planes, n, lt, pat_stride, pat, txt);
    *launches += 1;
    return cudaGetLastError();
}

}  // namespace tcrnet

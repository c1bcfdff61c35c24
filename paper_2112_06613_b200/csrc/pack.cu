// Step A1 (pack): validation, length histogram and the re-layout of the sequences into the two
// tables the distance kernel reads (residues "saved as a number ... BYTE";
// north_star subsystem (1): 5-bit residue codes, sorted by length, bucketed by length).
//
//   pat : one row per sorted position, one residue code (0..25) per byte, row stride
//         pat_stride bytes (multiple of 16), padded with 0xff - read once per work item to
//         build the Peq match masks.
//   txt : per length bucket, one row of round_up(len,4) 32-bit words per sequence holding the
//         residue code of each column, padded with kPadCode - streamed into shared memory
//         and read with one broadcast 128-bit load per four columns.  The code sits in a
//         32-bit word so that the per-column Peq address is a single IMAD (code * row_bytes
//         + lane offset) on the FMA pipe, leaving the ALU pipe to the bit-vector recurrence.
#include "tcrnet_internal.h"

namespace tcrnet {
namespace {

__global__ void __launch_bounds__(256) k_length_hist(const int32_t* __restrict__ lengths, int64_t n,
                                                    unsigned long long* __restrict__ hist,
                                                    uint32_t* __restrict__ flags) {
    __shared__ uint32_t h[kNumLen];
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

__global__ void __launch_bounds__(256) k_pack(const uint8_t* __restrict__ residues,
                                             const int64_t* __restrict__ offsets,
                                             const int32_t* __restrict__ lengths,
                                             const int32_t* __restrict__ perm, int64_t n,
                                             const __grid_constant__ LengthTable lt, int pat_stride,
                                             uint8_t* __restrict__ pat, uint32_t* __restrict__ txt,
                                             uint32_t* __restrict__ flags) {
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;  // sorted position
    bool bad = false;
    if (s < n) {
        const int32_t o = perm[s];
        const int32_t len = lengths[o];
        const uint8_t* src = residues + offsets[o];
        uint8_t* prow = pat + (size_t)s * pat_stride;
        uint32_t* trow = txt + lt.txt_base[len] + (int64_t)(s - lt.start[len]) * lt.row_words[len];
        const int rw = lt.row_words[len];
        for (int i = 0; i < pat_stride; ++i) {
            uint32_t c = 0xffu;
            if (i < len) {
                c = (uint32_t)src[i] - (uint32_t)'A';
                if (c >= (uint32_t)kNumCodes) {
                    bad = true;
                    c = 0;
                }
            }
            prow[i] = (uint8_t)c;
            if (i < rw) trow[i] = i < len ? c : (uint32_t)kPadCode;
        }
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(flags, kFlagBadResidue);
}

}  // namespace

cudaError_t launch_length_hist(const int32_t* lengths, int64_t n, unsigned long long* hist, uint32_t* flags,
                               cudaStream_t s, int* launches) {
    int64_t blocks = (n + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    k_length_hist<<<(unsigned)blocks, 256, 0, s>>>(lengths, n, hist, flags);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_pack(const uint8_t* residues, const int64_t* offsets, const int32_t* lengths,
                        const int32_t* perm, int64_t n, const LengthTable& lt, int pat_stride, uint8_t* pat,
                        uint32_t* txt, uint32_t* flags, cudaStream_t s, int* launches) {
    const int64_t blocks = (n + 255) / 256;
    k_pack<<<(unsigned)blocks, 256, 0, s>>>(residues, offsets, lengths, perm, n, lt, pat_stride, pat, txt, flags);
    *launches += 1;
    return cudaGetLastError();
}

}  // namespace tcrnet

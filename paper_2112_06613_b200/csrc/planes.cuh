// Bit-plane rows (written by pack.cu): sequence at sorted position s = 8 words of W; words 0..4 = planes (bit j of
// plane k = bit k of the 5-bit code of residue j, zero beyond the sequence), word 5 = length.  W = uint32_t when the
// set's longest sequence has <= 32 residues (32 bytes per row), else uint64_t.  Read by segjoin.cu and labels.cu.
#pragma once

#include "tcrnet_internal.h"

namespace tcrnet {
namespace {

template <typename W>
struct PlaneRow {
    W p[5];
    int len;
};

template <typename W>
__device__ __forceinline__ PlaneRow<W> load_planes(const void* __restrict__ planes, int64_t pos);
template <>
__device__ __forceinline__ PlaneRow<uint32_t> load_planes<uint32_t>(const void* __restrict__ planes, int64_t pos) {
    const uint4* row = reinterpret_cast<const uint4*>(planes) + 2 * pos;
    const uint4 a = __ldg(row), b = __ldg(row + 1);
    PlaneRow<uint32_t> r;
    r.p[0] = a.x, r.p[1] = a.y, r.p[2] = a.z, r.p[3] = a.w, r.p[4] = b.x;
    r.len = (int)b.y;
    return r;
}
template <>
__device__ __forceinline__ PlaneRow<uint64_t> load_planes<uint64_t>(const void* __restrict__ planes, int64_t pos) {
    const ulonglong2* row = reinterpret_cast<const ulonglong2*>(planes) + 4 * pos;
    const ulonglong2 a = __ldg(row), b = __ldg(row + 1), c = __ldg(row + 2);
    PlaneRow<uint64_t> r;
    r.p[0] = a.x, r.p[1] = a.y, r.p[2] = b.x, r.p[3] = b.y, r.p[4] = c.x;
    r.len = (int)c.y;
    return r;
}

}  // namespace
}  // namespace tcrnet

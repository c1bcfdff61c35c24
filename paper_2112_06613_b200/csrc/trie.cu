// Step A1, last part: the prefix trie over the sorted texts.
//
// Inside a length bucket the sequences are in lexicographic order of their first kSortPrefix
// residues (the sequence sort of tcrnet_load), so the texts that share their first k residues are
// consecutive.  Level k of the trie (k = 1..kTrieDepth) has one node per such run; the children of a
// level-k node are the level-(k+1) runs inside it (at most 27: one per distinct next residue code).
// The distance kernel of distance_trie.cu walks this trie once per warp of 32 patterns: the DP
// columns of a shared prefix are computed once per node instead of once per text, and a subtree
// whose prefix already proves lev > l_max for all 32 patterns is never entered (the exact early
// exit of PAPER.md:326, applied to a whole run of texts at once).
//
// Construction (all on the device, three streaming passes over N positions):
//   k_trie_lcp    lcp8[s] = number of leading residues sorted position s shares with s-1
//                 (0 at the first position of a bucket, kTrieDepth when >= kTrieDepth are shared);
//                 s starts a level-k run iff lcp8[s] < k.
//   k_trie_count  per tile of 1024 positions, the number of run starts of every level.
//   k_trie_scan   exclusive scan of the tile counts (one CTA), totals, sentinels.
//   k_trie_emit   node ids by ranking inside the tile; writes the nodes.
//   k_trie_child_codes  per node of levels 1..kTrieDepth-1, the bitmap of its children's residue codes
//                 (the guided expansion of distance_trie.cu addresses a child by popc(bitmap & low(code))).
#include "tcrnet_internal.h"

namespace tcrnet {
namespace {

constexpr int kThreads = 256;
constexpr int kItems = 4;                      // positions per thread: one 32-bit load of lcp8 (short serial chains:
                                               // these kernels are latency-bound at TCR scale)
constexpr int kTile = kThreads * kItems;       // 1024
constexpr int kCountStride = 8;                // uint32 per tile in tile_counts ([1..kTrieDepth] used)
static_assert(kTrieDepth <= 6, "level counts are packed as 4 x 16 bit + 2 x 16 bit");

// Length bucket of sorted position s: the largest L with start[L] <= s (empty buckets share their
// start with the next non-empty one, so this is the bucket that contains s).
__device__ __forceinline__ int bucket_of(const LengthTable& lt, int64_t s) {
    int lo = 0, hi = kNumLen;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (lt.start[mid] <= s) lo = mid; else hi = mid;
    }
    return lo;
}

__global__ void __launch_bounds__(kThreads) k_trie_lcp(const uint32_t* __restrict__ txt,
                                                      const __grid_constant__ LengthTable lt, int64_t n,
                                                      uint8_t* __restrict__ lcp8) {
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const int len = bucket_of(lt, s);
    const int64_t rel = s - lt.start[len];
    int lcp = 0;
    if (rel > 0) {
        const int rw = lt.row_words[len];
        const uint32_t* row = txt + lt.txt_base[len] + rel * rw;
        const uint32_t* prev = row - rw;
        const int lim = min(kTrieDepth, len);
        while (lcp < lim && row[lcp] == prev[lcp]) ++lcp;
        if (lcp == lim) lcp = kTrieDepth;  // past the end both rows are padding
    }
    lcp8[s] = (uint8_t)lcp;
}

// Run-start flags of one position packed as counters: level k in bits 16(k-1).. of lo (k = 1..4) and
// bits 16(k-5).. of hi (k = 5, 6).  A tile has 1024 positions, so 16 bits per counter suffice.
struct Packed {
    unsigned long long lo;
    uint32_t hi;
};
__device__ __forceinline__ Packed flags_of(uint32_t lcp) {
    Packed f{0ull, 0u};
#pragma unroll
    for (int k = 1; k <= kTrieDepth; ++k)
        if (lcp < (uint32_t)k) {
            if (k <= 4) f.lo += 1ull << (16 * (k - 1)); else f.hi += 1u << (16 * (k - 5));
        }
    return f;
}
__device__ __forceinline__ uint32_t level_count(const Packed& p, int k) {
    return k <= 4 ? (uint32_t)(p.lo >> (16 * (k - 1))) & 0xffffu : (p.hi >> (16 * (k - 5))) & 0xffffu;
}

// the kItems lcp values of this thread (255 = beyond n: starts nothing)
__device__ __forceinline__ void load_lcp16(const uint8_t* lcp8, int64_t first, int64_t n, uint32_t* v) {
    static_assert(kItems == 4, "one 32-bit load");
    const uint32_t w = *reinterpret_cast<const uint32_t*>(lcp8 + first);  // the buffer is padded to a multiple of 16
#pragma unroll
    for (int i = 0; i < kItems; ++i) v[i] = first + i < n ? (w >> (8 * i)) & 0xffu : 255u;
}

// Exclusive scan of one Packed per thread across the CTA; *total = CTA sum.
__device__ __forceinline__ Packed block_exclusive(Packed v, Packed* warp_sums /*[8]*/, Packed* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    Packed inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned long long ol = __shfl_up_sync(0xffffffffu, inc.lo, d);
        const uint32_t oh = __shfl_up_sync(0xffffffffu, inc.hi, d);
        if (lane >= d) {
            inc.lo += ol;
            inc.hi += oh;
        }
    }
    if (lane == 31) warp_sums[warp] = inc;
    __syncthreads();
    Packed before{0ull, 0u}, all{0ull, 0u};
#pragma unroll
    for (int w = 0; w < kThreads / 32; ++w) {
        const Packed ws = warp_sums[w];
        if (w < warp) {
            before.lo += ws.lo;
            before.hi += ws.hi;
        }
        all.lo += ws.lo;
        all.hi += ws.hi;
    }
    *total = all;
    return Packed{before.lo + inc.lo - v.lo, before.hi + inc.hi - v.hi};
}

__global__ void __launch_bounds__(kThreads) k_trie_count(const uint8_t* __restrict__ lcp8, int64_t n,
                                                        uint32_t* __restrict__ tile_counts) {
    __shared__ Packed ws[kThreads / 32];
    const int64_t first = (int64_t)blockIdx.x * kTile + (int64_t)threadIdx.x * kItems;
    Packed acc{0ull, 0u};
    if (first < n) {
        uint32_t v[kItems];
        load_lcp16(lcp8, first, n, v);
#pragma unroll
        for (int i = 0; i < kItems; ++i) {
            const Packed f = flags_of(v[i]);
            acc.lo += f.lo;
            acc.hi += f.hi;
        }
    }
    Packed total;
    block_exclusive(acc, ws, &total);
    if (threadIdx.x <= kTrieDepth && threadIdx.x >= 1)
        tile_counts[(size_t)blockIdx.x * kCountStride + threadIdx.x] = level_count(total, threadIdx.x);
}

// One CTA: tile_counts[tile][k] -> exclusive prefix over the tiles; counts[k] = total; sentinels.
__global__ void __launch_bounds__(1024) k_trie_scan(uint32_t* __restrict__ tile_counts, int64_t n_tiles, int64_t n,
                                                   const __grid_constant__ TrieLevels lv,
                                                   uint32_t* __restrict__ counts) {
    __shared__ uint32_t wsum[32];
    __shared__ uint32_t carry[kCountStride];
    __shared__ uint32_t chunk_total;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x < kCountStride) carry[threadIdx.x] = 0;
    __syncthreads();
    for (int64_t c = 0; c < n_tiles; c += 1024) {
        const int64_t t = c + threadIdx.x;
        for (int k = 1; k <= kTrieDepth; ++k) {
            const uint32_t v = t < n_tiles ? tile_counts[(size_t)t * kCountStride + k] : 0u;
            uint32_t inc = v;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t o = __shfl_up_sync(0xffffffffu, inc, d);
                if (lane >= d) inc += o;
            }
            if (lane == 31) wsum[warp] = inc;
            __syncthreads();
            if (warp == 0) {
                const uint32_t w = wsum[lane];
                uint32_t wi = w;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const uint32_t o = __shfl_up_sync(0xffffffffu, wi, d);
                    if (lane >= d) wi += o;
                }
                wsum[lane] = wi - w;
                if (lane == 31) chunk_total = wi;
            }
            __syncthreads();
            if (t < n_tiles) tile_counts[(size_t)t * kCountStride + k] = carry[k] + wsum[warp] + inc - v;
            __syncthreads();
            if (threadIdx.x == 0) carry[k] += chunk_total;
            __syncthreads();
        }
    }
    if (threadIdx.x >= 1 && threadIdx.x <= kTrieDepth) {
        const int k = threadIdx.x;
        counts[k] = carry[k];
        TrieNode sentinel;
        sentinel.text_begin = (uint32_t)n;
        sentinel.child_begin = k < kTrieDepth ? carry[k + 1] : (uint32_t)n;
        sentinel.code = (uint32_t)kPadCode;
        sentinel.child_codes = 0u;
        lv.p[k][carry[k]] = sentinel;
    }
}

__global__ void __launch_bounds__(kThreads) k_trie_emit(const uint32_t* __restrict__ txt,
                                                       const __grid_constant__ LengthTable lt, int64_t n,
                                                       const uint8_t* __restrict__ lcp8,
                                                       const uint32_t* __restrict__ tile_base,
                                                       const __grid_constant__ TrieLevels lv,
                                                       uint32_t* __restrict__ root) {
    __shared__ Packed ws[kThreads / 32];
    __shared__ TrieNode* level_nodes[kTrieDepth + 1];
    __shared__ uint32_t base[kCountStride];
    if (threadIdx.x <= kTrieDepth) {
        level_nodes[threadIdx.x] = lv.p[threadIdx.x];
        base[threadIdx.x] = threadIdx.x >= 1 ? tile_base[(size_t)blockIdx.x * kCountStride + threadIdx.x] : 0u;
    }
    const int64_t first = (int64_t)blockIdx.x * kTile + (int64_t)threadIdx.x * kItems;
    uint32_t v[kItems];
    Packed acc{0ull, 0u};
    if (first < n) {
        load_lcp16(lcp8, first, n, v);
#pragma unroll
        for (int i = 0; i < kItems; ++i) {
            const Packed f = flags_of(v[i]);
            acc.lo += f.lo;
            acc.hi += f.hi;
        }
    }
    Packed total;
    Packed run = block_exclusive(acc, ws, &total);  // run starts of this tile before this thread (has a barrier)
    if (first >= n) return;
    uint32_t id[kTrieDepth + 2];
#pragma unroll
    for (int k = 1; k <= kTrieDepth; ++k) id[k] = base[k] + level_count(run, k);
    int len = bucket_of(lt, first);
    for (int i = 0; i < kItems; ++i) {
        const int64_t s = first + i;
        if (s >= n) break;
        const uint32_t lcp = v[i];
        if (lcp >= (uint32_t)kTrieDepth) continue;  // starts no run
        while (s >= lt.start[len + 1]) ++len;
        const uint32_t* row = txt + lt.txt_base[len] + (s - lt.start[len]) * lt.row_words[len];
        if (s == lt.start[len]) root[len] = id[1];
        id[kTrieDepth + 1] = (uint32_t)s;  // the "children" of the deepest level are the texts themselves
#pragma unroll
        for (int k = 1; k <= kTrieDepth; ++k) {
            if (lcp < (uint32_t)k) {
                TrieNode nd;
                nd.text_begin = (uint32_t)s;
                nd.child_begin = id[k + 1];
                nd.code = k - 1 < len ? row[k - 1] : (uint32_t)kPadCode;
                nd.child_codes = 0u;
                level_nodes[k][id[k]] = nd;
            }
        }
#pragma unroll
        for (int k = 1; k <= kTrieDepth; ++k)
            if (lcp < (uint32_t)k) ++id[k];
    }
}

// blockIdx.y + 1 = level k; thread = node of level k; OR of the codes of its children in level k+1.
__global__ void __launch_bounds__(kThreads) k_trie_child_codes(const __grid_constant__ TrieLevels lv,
                                                              const uint32_t* __restrict__ counts) {
    const int k = blockIdx.y + 1;
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= counts[k]) return;
    TrieNode* nodes = lv.p[k];
    const TrieNode* kids = lv.p[k + 1];
    const uint32_t b = nodes[i].child_begin, e = nodes[i + 1].child_begin;  // i + 1 may be the sentinel
    uint32_t codes = 0u;
    for (uint32_t c = b; c < e; ++c) codes |= 1u << (kids[c].code & 31u);
    nodes[i].child_codes = codes;
}

}  // namespace

int64_t trie_tiles(int64_t n) { return n > 0 ? (n + kTile - 1) / kTile : 1; }

int64_t trie_level_capacity(int64_t n, int level) {
    // at most 27 children per node, one root set per length bucket; never more nodes than texts
    int64_t cap = kNumLen;
    for (int k = 0; k < level && cap < n; ++k) cap *= 27;
    return (cap < n ? cap : n) + 1;  // + sentinel
}

cudaError_t launch_trie_build(const uint32_t* txt, const LengthTable& lt, int64_t n, uint8_t* lcp8,
                              uint32_t* tile_counts, const TrieLevels& lv, uint32_t* counts, uint32_t* root,
                              cudaStream_t s, int* launches) {
    const int64_t tiles = trie_tiles(n);
    k_trie_lcp<<<(unsigned)((n + kThreads - 1) / kThreads), kThreads, 0, s>>>(txt, lt, n, lcp8);
    k_trie_count<<<(unsigned)tiles, kThreads, 0, s>>>(lcp8, n, tile_counts);
    k_trie_scan<<<1, 1024, 0, s>>>(tile_counts, tiles, n, lv, counts);
    k_trie_emit<<<(unsigned)tiles, kThreads, 0, s>>>(txt, lt, n, lcp8, tile_counts, lv, root);
    k_trie_child_codes<<<dim3((unsigned)((n + kThreads - 1) / kThreads), kTrieDepth - 1), kThreads, 0, s>>>(lv, counts);
    *launches += 5;
    return cudaGetLastError();
}

}  // namespace tcrnet

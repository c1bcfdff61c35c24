// Step A0 (before the pack): rows with identical sequences are collapsed.
//
// Reading Q3 keeps one node per input row, and repertoires are full of repeated CDR3
// sequences (public clones).  Identical rows have identical distances to everything,
// so the all-pairs step runs over the DISTINCT sequences only and the emission multiplies a surviving
// pair of distinct sequences by the rows behind them (myers.cuh emit_edges); the rows of one sequence
// are joined to each other directly (k_emit_cliques: d = 0 <= l_max for every l_max).  Nothing about
// the result changes - only the number of pairs the distance kernel has to decide.
//
//   k_dedup_insert   open-addressing table, one 64-bit word per slot = (fingerprint << 32) | smallest row
//                    seen with that fingerprint: atomicCAS on the empty slot, atomicMin afterwards
//   k_dedup_lookup   every row finds its slot again, compares its bytes with the slot's row and becomes a
//                    duplicate of it, or (first row of its sequence, fingerprint clash, invalid row) stays
//   scan             ids of the distinct sequences in input-row order (deterministic)
//   k_dedup_groups   uid of every row, rows per uid, length / residue offset of every uid
//   scan + k_dedup_fill   the rows of every uid, contiguous (order inside a group is irrelevant); total clique edges
// Rows with an invalid length or out-of-range offset are never read and never merged; the pack step
// reports them.  HBM/L2-bound: ~100 B per row over all kernels.
#include "launch.cuh"
#include "tcrnet_internal.h"

namespace tcrnet {
namespace {

constexpr unsigned long long kEmptySlot = ~0ull;

__device__ __forceinline__ bool row_ok(int64_t off, int32_t len, int64_t total_len) {
    return len >= 1 && len <= kMaxLen && off >= 0 && off + len <= total_len;
}

__device__ __forceinline__ unsigned long long hash_row(const uint8_t* src, int len) {
    unsigned long long h = 0xcbf29ce484222325ull ^ (unsigned long long)len;
    for (int i = 0; i < len; ++i) h = (h ^ src[i]) * 0x100000001b3ull;  // FNV-1a
    h ^= h >> 33;                                                      // + a finaliser for the high bits
    h *= 0xff51afd7ed558ccdull;
    h ^= h >> 33;
    return h;
}

// The probe path of a row starts at a slot derived from its FINGERPRINT alone, so all rows with one fingerprint walk
// the same path and meet in one slot whatever the order of the inserts: which rows collapse does not depend on timing
// (two different sequences with one fingerprint: the rows of the one that owns the smallest row collapse, the rows of
// the other stay sequences of their own - on every rank of a sharded build alike).
__device__ __forceinline__ uint32_t start_slot(unsigned long long fp, uint32_t mask) {
    return (uint32_t)(((fp >> 32) * 0x9E3779B97F4A7C15ull) >> 32) & mask;
}

// Also the length histogram of the ROWS and their validation (what k_length_hist does for a load without collapse):
// the lengths are read here anyway.
__global__ void __launch_bounds__(256) k_dedup_insert(const uint8_t* __restrict__ residues,
                                                     const int64_t* __restrict__ offsets,
                                                     const int32_t* __restrict__ lengths, int64_t n, int64_t total_len,
                                                     unsigned long long* __restrict__ table, uint32_t mask,
                                                     unsigned long long* __restrict__ hash,
                                                     unsigned long long* __restrict__ hist, uint32_t* __restrict__ flags) {
    grid_dependency_wait();
    __shared__ uint32_t h[kNumLen];
    for (int k = threadIdx.x; k < kNumLen; k += blockDim.x) h[k] = 0;
    __syncthreads();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool bad = false;
    if (i < n) {
        const int64_t off = offsets[i];
        const int32_t len = lengths[i];
        bad = len < 1 || len > kMaxLen;
        atomicAdd(&h[bad ? 0 : len], 1u);
        if (!row_ok(off, len, total_len)) {
            hash[i] = kEmptySlot;  // never merged
        } else {
            unsigned long long hv = hash_row(residues + off, len);
            if (hv == kEmptySlot) hv = 0;
            hash[i] = hv;
            const unsigned long long fp = hv & 0xffffffff00000000ull;
            const unsigned long long mine = fp | (unsigned long long)i;
            uint32_t s = start_slot(fp, mask);
            for (;;) {
                unsigned long long cur = table[s];
                if (cur == kEmptySlot) {
                    cur = atomicCAS(&table[s], kEmptySlot, mine);
                    if (cur == kEmptySlot) break;
                }
                if ((cur & 0xffffffff00000000ull) == fp) {
                    atomicMin(&table[s], mine);
                    break;
                }
                s = (s + 1u) & mask;
            }
        }
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(flags, kFlagBadLength);
    for (int k = threadIdx.x; k < kNumLen; k += blockDim.x)
        if (h[k]) atomicAdd(&hist[k], (unsigned long long)h[k]);
}

__global__ void __launch_bounds__(256) k_dedup_lookup(const uint8_t* __restrict__ residues,
                                                     const int64_t* __restrict__ offsets,
                                                     const int32_t* __restrict__ lengths, int64_t n,
                                                     const unsigned long long* __restrict__ table, uint32_t mask,
                                                     const unsigned long long* __restrict__ hash,
                                                     int32_t* __restrict__ rep_of, uint32_t* __restrict__ is_first) {
    grid_dependency_wait();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const unsigned long long h = hash[i];
    int64_t rep = i;
    if (h != kEmptySlot) {
        const unsigned long long fp = h & 0xffffffff00000000ull;
        uint32_t s = start_slot(fp, mask);
        for (;;) {
            const unsigned long long cur = table[s];
            if ((cur & 0xffffffff00000000ull) == fp && cur != kEmptySlot) {
                rep = (int64_t)(cur & 0xffffffffull);
                break;
            }
            s = (s + 1u) & mask;
        }
        if (rep != i) {
            const int32_t len = lengths[i];
            bool same = lengths[rep] == len;
            if (same) {
                const uint8_t* a = residues + offsets[i];
                const uint8_t* b = residues + offsets[rep];
                for (int k = 0; k < len; ++k) same = same && a[k] == b[k];
            }
            if (!same) rep = i;  // fingerprint clash: stays a sequence of its own
        }
    }
    rep_of[i] = (int32_t)rep;
    is_first[i] = rep == i ? 1u : 0u;
}

__global__ void __launch_bounds__(256) k_dedup_groups(const int32_t* __restrict__ rep_of,
                                                     const uint32_t* __restrict__ first_rank,
                                                     const int64_t* __restrict__ offsets,
                                                     const int32_t* __restrict__ lengths, int64_t n,
                                                     int32_t* __restrict__ uid_of, uint32_t* __restrict__ group_count,
                                                     int32_t* __restrict__ len_u, int64_t* __restrict__ off_u,
                                                     unsigned long long* __restrict__ hist_u,
                                                     unsigned long long* __restrict__ sort_key,
                                                     int32_t* __restrict__ sort_val) {
    grid_dependency_wait();
    __shared__ uint32_t h[kNumLen];  // length histogram of the distinct sequences (their first rows)
    for (int k = threadIdx.x; k < kNumLen; k += blockDim.x) h[k] = 0;
    __syncthreads();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        const int32_t rep = rep_of[i];
        const uint32_t uid = first_rank[rep];
        uid_of[i] = (int32_t)uid;
        atomicAdd(&group_count[uid], 1u);
        if (rep == i) {
            const int32_t len = lengths[i];
            len_u[uid] = len;
            off_u[uid] = offsets[i];
            const int l = (len < 1 || len > kMaxLen) ? 0 : len;
            atomicAdd(&h[l], 1u);
            // (a load that is bucketed by length only: the key k_seq_keys would write, without its residue digits)
            if (sort_key) sort_key[uid] = (unsigned long long)(uint32_t)(l > 0 ? l - 1 : 0) << (5 * kSortPrefix), sort_val[uid] = (int32_t)uid;
        }
    }
    __syncthreads();
    for (int k = threadIdx.x; k < kNumLen; k += blockDim.x)
        if (h[k]) atomicAdd(&hist_u[k], (unsigned long long)h[k]);
}

// group_count[uid] counts down to 0 while the rows take their places
// (the row that takes the last free slot also adds the group's g (g - 1) / 2 clique edges to *clique_edges: a load
// dominated by one heavily repeated sequence can then be refused before any quadratic work is done)
__global__ void __launch_bounds__(256) k_dedup_fill(const int32_t* __restrict__ uid_of, int64_t n,
                                                   const uint32_t* __restrict__ group_start,
                                                   uint32_t* __restrict__ group_count, int32_t* __restrict__ members,
                                                   unsigned long long* __restrict__ clique_edges,
                                                   uint32_t* __restrict__ max_group) {
    grid_dependency_wait();
    __shared__ unsigned long long block_sum;
    __shared__ uint32_t block_max;
    if (threadIdx.x == 0) block_sum = 0ull, block_max = 0u;
    __syncthreads();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long mine = 0ull;
    uint32_t g_mine = 0u;
    if (i < n) {
        const uint32_t uid = (uint32_t)uid_of[i];
        const uint32_t slot = atomicSub(&group_count[uid], 1u) - 1u;
        const uint32_t b = group_start[uid];
        members[b + slot] = (int32_t)i;
        if (slot == 0u) {
            const unsigned long long g = group_start[uid + 1u] - b;
            mine = g * (g - 1ull) / 2ull;
            g_mine = (uint32_t)g;
        }
    }
    // ... and the largest group: the expansion of the recorded pairs needs its second kernel only if two groups can
    // have more than kHuge pairs of rows between them
    g_mine = __reduce_max_sync(0xffffffffu, g_mine);
    if ((threadIdx.x & 31) == 0 && g_mine > 1u) atomicMax(&block_max, g_mine);
    // one atomic per CTA on the global sum (one per shared sequence on a single address cost 40 us at config 4)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_xor_sync(0xffffffffu, mine, o);
    if ((threadIdx.x & 31) == 0 && mine) atomicAdd(&block_sum, mine);
    __syncthreads();
    if (threadIdx.x == 0 && block_sum) atomicAdd(clique_edges, block_sum);
    if (threadIdx.x == 0 && block_max) atomicMax(max_group, block_max);
}

// Edges between the rows of one sequence: the thread of member slot x joins it to the slots after it.  Output
// offsets: warp scan + one atomicAdd per warp.  Counting for the CSR step is done per ROW, not per edge: row r
// of a group has one edge to every other row of it, the larger ones count for row_count[r], the smaller for deg[r].
__global__ void __launch_bounds__(256) k_emit_cliques(const int32_t* __restrict__ members,
                                                     const int32_t* __restrict__ uid_of,
                                                     const uint32_t* __restrict__ group_start, int64_t n,
                                                     unsigned long long* __restrict__ edges,
                                                     unsigned long long* __restrict__ edge_count,
                                                     unsigned long long edge_cap, int32_t* __restrict__ row_count,
                                                     int32_t* __restrict__ deg, uint32_t shard, uint32_t n_shards) {
    grid_dependency_wait();
    constexpr uint32_t kFullMask = 0xffffffffu;
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    uint32_t r = 0, begin = 0, end = 0, rest = 0;
    if (s < n) {
        r = (uint32_t)members[s];
        const uint32_t uid = (uint32_t)uid_of[r];
        if (uid % n_shards == shard) {  // step 8(e): the shared sequences are dealt out to the shards by uid
            begin = group_start[uid];
            end = group_start[uid + 1u];
            rest = end - 1u - (uint32_t)s;  // slots after this one
        }
    }
    if (end - begin > 1u) {
        uint32_t larger = 0;
        for (uint32_t y = begin; y < end; ++y) larger += (uint32_t)members[y] > r;
        const uint32_t smaller = end - begin - 1u - larger;
        if (larger) atomicAdd(row_count + r, (int)larger);
        if (smaller) atomicAdd(deg + r, (int)smaller);
    }
    if (!__any_sync(kFullMask, rest != 0u)) return;
    unsigned long long incl = rest;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long v = __shfl_up_sync(kFullMask, incl, o);
        if (lane >= o) incl += v;
    }
    unsigned long long base = 0;
    if (lane == 31) base = atomicAdd(edge_count, incl);
    unsigned long long pos = __shfl_sync(kFullMask, base, 31) + incl - rest;
    for (uint32_t y = (uint32_t)s + 1u; y < end; ++y, ++pos) {
        const uint32_t q = (uint32_t)members[y];
        const uint32_t a = min(r, q), b = max(r, q);
        if (pos < edge_cap) edges[pos] = ((unsigned long long)a << 32) | b;
    }
}

// The pairs of distinct sequences the distance kernel recorded (codes: a row, or kGroupFlag | uid) -> the edges
// between the rows behind them, counted for the CSR step.  One warp handles 32 entries: the output offsets are
// a warp scan + one atomicAdd; a lane writes up to kOwn edges itself, larger products are shared by the warp.
__global__ void __launch_bounds__(256) k_expand_entries(const unsigned long long* __restrict__ entries,
                                                       const unsigned long long* __restrict__ n_entries_dev,
                                                       unsigned long long entry_cap,
                                                       const uint32_t* __restrict__ group_start,
                                                       const int32_t* __restrict__ members,
                                                       unsigned long long* __restrict__ edges,
                                                       unsigned long long* __restrict__ edge_total,
                                                       unsigned long long edge_cap, int32_t* __restrict__ row_count,
                                                       int32_t* __restrict__ deg, ulonglong2* __restrict__ huge,
                                                       unsigned long long* __restrict__ n_huge, uint32_t huge_cap) {
    grid_dependency_wait();
    constexpr uint32_t kFullMask = 0xffffffffu;
    constexpr unsigned long long kOwn = 8;
    constexpr unsigned long long kHuge = 4096;  // products beyond this are left to k_expand_huge (the whole grid)
    const unsigned long long n_ent = min(*n_entries_dev, entry_cap);
    const int lane = threadIdx.x & 31;
    const unsigned long long warps = ((unsigned long long)gridDim.x * blockDim.x) >> 5;
    for (unsigned long long e0 = ((unsigned long long)blockIdx.x * blockDim.x + threadIdx.x) & ~31ull; e0 < n_ent;
         e0 += warps * 32ull) {
        const bool have = e0 + lane < n_ent;
        const unsigned long long key = have ? entries[e0 + lane] : 0ull;
        const uint32_t oi = (uint32_t)(key >> 32), oj = (uint32_t)key;
        uint32_t bi = 0, ni = 1, bj = 0, nj = 1;  // rows behind each side: members[b .. b + n), or the row itself
        if (have && (oi & kGroupFlag)) {
            const uint32_t g = oi & ~kGroupFlag;
            bi = group_start[g];
            ni = group_start[g + 1] - bi;
        }
        if (have && (oj & kGroupFlag)) {
            const uint32_t g = oj & ~kGroupFlag;
            bj = group_start[g];
            nj = group_start[g + 1] - bj;
        }
        const unsigned long long w = have ? (unsigned long long)ni * nj : 0ull;
        unsigned long long incl = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long v = __shfl_up_sync(kFullMask, incl, o);
            if (lane >= o) incl += v;
        }
        unsigned long long base = 0;
        if (lane == 31) base = atomicAdd(edge_total, incl);
        base = __shfl_sync(kFullMask, base, 31);
        const unsigned long long first = base + incl - w;
        auto put = [&](unsigned long long pos, uint32_t ri, uint32_t rj) {
            const uint32_t a = min(ri, rj), b = max(ri, rj);
            atomicAdd(row_count + a, 1);
            atomicAdd(deg + b, 1);
            if (pos < edge_cap) edges[pos] = ((unsigned long long)a << 32) | b;
        };
        if (have && w <= kOwn) {
            unsigned long long pos = first;
            for (uint32_t x = 0; x < ni; ++x) {
                const uint32_t ri = (oi & kGroupFlag) ? (uint32_t)members[bi + x] : oi;
                for (uint32_t y = 0; y < nj; ++y, ++pos) put(pos, ri, (oj & kGroupFlag) ? (uint32_t)members[bj + y] : oj);
            }
        }
        uint32_t big = __ballot_sync(kFullMask, have && w > kOwn);
        while (big) {
            const int src = __ffs((int)big) - 1;
            big &= big - 1u;
            const uint32_t s_oi = __shfl_sync(kFullMask, oi, src), s_oj = __shfl_sync(kFullMask, oj, src);
            const uint32_t s_bi = __shfl_sync(kFullMask, bi, src), s_bj = __shfl_sync(kFullMask, bj, src);
            const uint32_t s_nj = __shfl_sync(kFullMask, nj, src);
            const unsigned long long s_w = __shfl_sync(kFullMask, w, src), s_first = __shfl_sync(kFullMask, first, src);
            if (s_w > kHuge) {  // two heavily repeated sequences: one warp would take milliseconds
                unsigned long long slot = 0;
                if (lane == 0) slot = atomicAdd(n_huge, 1ull);
                slot = __shfl_sync(kFullMask, slot, 0);
                if (slot < huge_cap) {
                    if (lane == 0) huge[slot] = make_ulonglong2(((unsigned long long)s_oi << 32) | s_oj, s_first);
                    continue;
                }
            }
            // (x, y) = (k / nj, k % nj) kept incrementally: one 32-bit division per lane and product instead of a
            // 64-bit one per edge
            uint32_t x = (uint32_t)lane / s_nj, y = (uint32_t)lane % s_nj;
            const uint32_t dx = 32u / s_nj, dy = 32u % s_nj;
            for (unsigned long long k = (unsigned long long)lane; k < s_w; k += 32ull) {
                put(s_first + k, (s_oi & kGroupFlag) ? (uint32_t)members[s_bi + x] : s_oi,
                    (s_oj & kGroupFlag) ? (uint32_t)members[s_bj + y] : s_oj);
                x += dx;
                y += dy;
                if (y >= s_nj) y -= s_nj, ++x;
            }
        }
    }
}

// The products k_expand_entries set aside (both sequences repeated so often that rows x rows > kHuge): every product
// is spread over the whole grid.
__global__ void __launch_bounds__(256) k_expand_huge(const ulonglong2* __restrict__ huge,
                                                    const unsigned long long* __restrict__ n_huge, uint32_t huge_cap,
                                                    const uint32_t* __restrict__ group_start,
                                                    const int32_t* __restrict__ members,
                                                    unsigned long long* __restrict__ edges, unsigned long long edge_cap,
                                                    int32_t* __restrict__ row_count, int32_t* __restrict__ deg) {
    grid_dependency_wait();
    const unsigned long long cnt = min(*n_huge, (unsigned long long)huge_cap);
    const unsigned long long tid = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long h = 0; h < cnt; ++h) {
        const ulonglong2 it = huge[h];
        const uint32_t oi = (uint32_t)(it.x >> 32), oj = (uint32_t)it.x;
        uint32_t bi = 0, ni = 1, bj = 0, nj = 1;
        if (oi & kGroupFlag) {
            const uint32_t g = oi & ~kGroupFlag;
            bi = group_start[g];
            ni = group_start[g + 1] - bi;
        }
        if (oj & kGroupFlag) {
            const uint32_t g = oj & ~kGroupFlag;
            bj = group_start[g];
            nj = group_start[g + 1] - bj;
        }
        const unsigned long long w = (unsigned long long)ni * nj;
        for (unsigned long long k = tid; k < w; k += stride) {
            const uint32_t x = (uint32_t)(k / nj), y = (uint32_t)(k % nj);
            const uint32_t ri = (oi & kGroupFlag) ? (uint32_t)members[bi + x] : oi;
            const uint32_t rj = (oj & kGroupFlag) ? (uint32_t)members[bj + y] : oj;
            const uint32_t a = min(ri, rj), b = max(ri, rj);
            atomicAdd(row_count + a, 1);
            atomicAdd(deg + b, 1);
            const unsigned long long pos = it.y + k;
            if (pos < edge_cap) edges[pos] = ((unsigned long long)a << 32) | b;
        }
    }
}

// inverse of the coded perm: every row -> the sorted position of its sequence
__global__ void __launch_bounds__(256) k_inverse_perm_groups(const int32_t* __restrict__ perm, int64_t n_u,
                                                            const uint32_t* __restrict__ group_start,
                                                            const int32_t* __restrict__ members,
                                                            int32_t* __restrict__ inv) {
    grid_dependency_wait();
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_u) return;
    const uint32_t code = (uint32_t)perm[s];
    if (code & kGroupFlag) {
        const uint32_t uid = code & ~kGroupFlag;
        for (uint32_t k = group_start[uid]; k < group_start[uid + 1]; ++k) inv[members[k]] = (int32_t)s;
    } else {
        inv[code] = (int32_t)s;
    }
}

unsigned grid_for(int64_t n) { return (unsigned)((n + 255) / 256); }

}  // namespace

uint32_t dedup_table_slots(int64_t n) {
    uint32_t m = 1024;
    while ((int64_t)m < 2 * n && m < (1u << 31)) m <<= 1;
    return m;
}

cudaError_t launch_dedup_find(const uint8_t* residues, const int64_t* offsets, const int32_t* lengths, int64_t n,
                              int64_t total_len, unsigned long long* table, uint32_t slots, unsigned long long* hash,
                              int32_t* rep_of, uint32_t* is_first, unsigned long long* hist, uint32_t* flags,
                              cudaStream_t s, int* launches) {
    // (table is all ones: cleared by the caller, ahead of the kernels that precede this one)
    launch_dep(k_dedup_insert, grid_for(n), 256, 0, s, residues, offsets, lengths, n, total_len, table, slots - 1u,
               hash, hist, flags);
    launch_dep(k_dedup_lookup, grid_for(n), 256, 0, s, residues, offsets, lengths, n, table, slots - 1u, hash, rep_of,
               is_first);
    *launches += 2;
    return cudaGetLastError();
}

cudaError_t launch_dedup_groups(const int32_t* rep_of, const uint32_t* first_rank, const int64_t* offsets,
                                const int32_t* lengths, int64_t n, int32_t* uid_of, uint32_t* group_count,
                                int32_t* len_u, int64_t* off_u, unsigned long long* hist_u,
                                unsigned long long* sort_key, int32_t* sort_val, cudaStream_t s, int* launches) {
    launch_dep(k_dedup_groups, grid_for(n), 256, 0, s, rep_of, first_rank, offsets, lengths, n, uid_of, group_count,
               len_u, off_u, hist_u, sort_key, sort_val);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_dedup_fill(const int32_t* uid_of, int64_t n, const uint32_t* group_start, uint32_t* group_count,
                              int32_t* members, unsigned long long* clique_edges, uint32_t* max_group, cudaStream_t s,
                              int* launches) {
    launch_dep(k_dedup_fill, grid_for(n), 256, 0, s, uid_of, n, group_start, group_count, members, clique_edges,
               max_group);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_emit_cliques(const int32_t* members, const int32_t* uid_of, const uint32_t* group_start, int64_t n,
                                unsigned long long* edges, unsigned long long* edge_count, unsigned long long edge_cap,
                                int32_t* row_count, int32_t* deg, int shard, int n_shards, cudaStream_t s, int* launches) {
    launch_dep(k_emit_cliques, grid_for(n), 256, 0, s, members, uid_of, group_start, n, edges, edge_count, edge_cap, row_count, deg,
                                               (uint32_t)shard, (uint32_t)n_shards);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_expand_entries(const unsigned long long* entries, const unsigned long long* n_entries_dev,
                                  unsigned long long entry_cap, const uint32_t* group_start, const int32_t* members,
                                  unsigned long long* edges, unsigned long long* edge_total, unsigned long long edge_cap,
                                  int32_t* row_count, int32_t* deg, void* huge, unsigned long long* n_huge,
                                  uint32_t huge_cap, bool huge_possible, int n_sm, cudaStream_t s, int* launches) {
    launch_dep(k_expand_entries, (unsigned)(n_sm * 8), 256, 0, s, entries, n_entries_dev, entry_cap, group_start, members, edges,
                                                          edge_total, edge_cap, row_count, deg, (ulonglong2*)huge, n_huge,
                                                          huge_possible ? huge_cap : 0u);  // (0: nothing is set aside)
    *launches += 1;
    if (!huge_possible) return cudaGetLastError();  // (no two groups of the load have more than kHuge pairs of rows)
    launch_dep(k_expand_huge, (unsigned)(n_sm * 8), 256, 0, s, (const ulonglong2*)huge, n_huge, huge_cap, group_start, members,
                                                       edges, edge_cap, row_count, deg);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_inverse_perm_groups(const int32_t* perm, int64_t n_u, const uint32_t* group_start,
                                       const int32_t* members, int32_t* inv, cudaStream_t s, int* launches) {
    launch_dep(k_inverse_perm_groups, grid_for(n_u), 256, 0, s, perm, n_u, group_start, members, inv);
    *launches += 1;
    return cudaGetLastError();
}

}  // namespace tcrnet

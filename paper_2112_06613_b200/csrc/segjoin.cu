// Segment join: an exact candidate filter in front of steps A3-A5 (the tile scheduler of north_star (2) taken one
// step further: not only length-bucket pairs that cannot match are skipped, but every pair that shares no segment).
//
// Pigeonhole: cut a text s (length n) into k = l_max + 1 consecutive segments.  An edit script of at most l_max
// operations touches at most l_max of them, so if lev(r, s) <= l_max at least one segment of s
// occurs UNCHANGED in r.  Take the first such segment, number i, starting at p in s and found at p + d in r
// (delta = n - |r| >= 0: the pattern r is the shorter sequence).  Each of the i segments before it holds at least
// one edit, the part before the match needs at least |d| insertions / deletions and the part after it at least
// |d + delta|, so   max(|d|, i) + |d + delta| <= l_max.   These (i, d) are the probes of JoinTables; everything else
// cannot be the first unchanged segment of a pair within l_max.  The filter has no false negatives; what it lets
// through is decided exactly, by the same column recurrence as everywhere else (myers.cuh) or - l_max <= 1, the
// fast path of SURVEY 8(f) NEXT-4 - by XOR / popcount on the 5-bit packed codes.
//
//   index   k_join_count / k_join_fill: one entry (tag, text) per (text, segment), bucketed by a hash of
//           (n, i, segment residues) in a power-of-two directory (count -> prefix sum -> fill).
//   probe   one lane = one pattern: for every text length n = m .. m + l_max and every probe (i, d) it hashes its own
//           residues [p + d, p + d + len), walks the directory bucket and queues the texts whose tag matches (same
//           length bucket: only texts after the pattern in sorted order, so every unordered pair is seen once).
//   verify  k_join: whenever a lane's queue is full (and at the end) the warp runs the recurrence in lock step, each
//           lane on its own candidate with its own Peq column (layout Peq[code][lane]: conflict-free), text residues
//           from the candidate's 5-bit row held in registers, the final-diagonal cell tracked from D0 as in the trie
//           kernel, one exit vote per column.  k_join_l1: the check is inline (no Peq, no queue).
//   once    a pair can be found through several probes.  It is emitted by the FIRST probe (in table order) whose
//           segment matches residue by residue - hash collisions never emit, true pairs emit exactly once.
#include <algorithm>

#include "myers.cuh"

namespace tcrnet {
namespace {

constexpr uint32_t kFullMask = 0xffffffffu;
constexpr int kJoinWarps = 8;
constexpr int kJoinThreads = 32 * kJoinWarps;
constexpr int kJoinQueue = 8;        // candidates a lane collects before the warp verifies
constexpr int kJoinDead = 1 << 20;   // dg of a lane without a candidate

// bits [pos, pos + nbits), nbits <= 32, of a row of 32-bit words (the word after the row may be read: the table
// is allocated with slack)
__device__ __forceinline__ uint32_t row_bits(const uint32_t* __restrict__ row, int pos, int nbits) {
    const int w = pos >> 5, sh = pos & 31;
    const uint32_t v = __funnelshift_r(__ldg(row + w), __ldg(row + w + 1), sh);
    return nbits >= 32 ? v : (v & ((1u << nbits) - 1u));
}

// hash of (text length n, segment i, residues [q, q + len) of `row`)
__device__ __forceinline__ unsigned long long seg_hash(const uint32_t* __restrict__ row, int q, int len, int n, int i) {
    unsigned long long h = 0x9E3779B97F4A7C15ull ^ ((unsigned long long)(n * 8 + i) * 0xD6E8FEB86659FD93ull);
    int pos = 5 * q, bits = 5 * len;
    while (bits > 0) {
        const int nb = min(bits, 30);  // six residues at a time
        h = (h ^ row_bits(row, pos, nb)) * 0xFF51AFD7ED558CCDull;
        h ^= h >> 32;
        pos += nb;
        bits -= nb;
    }
    h *= 0xC4CEB9FE1A85EC53ull;
    h ^= h >> 29;
    return h;
}

__device__ __forceinline__ bool seg_equal(const uint32_t* __restrict__ a, int qa, const uint32_t* __restrict__ b, int qb,
                                          int len) {
    int pa = 5 * qa, pb = 5 * qb, bits = 5 * len;
    while (bits > 0) {
        const int nb = min(bits, 30);
        if (row_bits(a, pa, nb) != row_bits(b, pb, nb)) return false;
        pa += nb;
        pb += nb;
        bits -= nb;
    }
    return true;
}

__device__ __forceinline__ int length_of(const LengthTable& lt, int64_t t) {  // bucket of sorted position t
    int lo = 0, hi = kNumLen;  // start[lo] <= t < start[hi]
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if ((int64_t)lt.start[mid] <= t) lo = mid; else hi = mid;
    }
    return lo;
}

// ---- index ----
template <bool FILL>
__global__ void __launch_bounds__(256) k_join_index(const uint32_t* __restrict__ seq5, int s5_words,
                                                   const __grid_constant__ LengthTable lt, int64_t n,
                                                   const __grid_constant__ JoinTables tab, uint32_t* __restrict__ cnt,
                                                   const uint32_t* __restrict__ dir, uint2* __restrict__ entries,
                                                   uint32_t mask) {
    const int k = tab.n_seg;
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t t = idx / k;
    const int i = (int)(idx - t * k);
    if (t >= n) return;
    const int len_t = length_of(lt, t);
    if (len_t < k) return;  // too short to be cut into k segments: such buckets stay with the other kernels
    const int q = tab.seg_start[len_t][i], len = tab.seg_start[len_t][i + 1] - q;
    const unsigned long long h = seg_hash(seq5 + (size_t)t * s5_words, q, len, len_t, i);
    const uint32_t b = (uint32_t)h & mask;
    if (!FILL) {
        atomicAdd(cnt + b, 1u);
    } else {
        const uint32_t slot = atomicSub(cnt + b, 1u) - 1u;
        entries[dir[b] + slot] = make_uint2((uint32_t)(h >> 32), (uint32_t)t);
    }
}

// ---- shared by the two join kernels ----
struct JoinParams {
    DistanceParams d;  // emission, queue, n_items, shard
    const JoinRow* rows;
    int32_t n_rows;
    int32_t s5_words;
    const uint32_t* seq5;
    JoinIndex index;
    JoinTables tab;
};

__device__ __forceinline__ const JoinRow& find_join_row(const JoinParams& S, int64_t item) {
    int lo = 0, hi = S.n_rows;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (S.rows[mid].item_begin <= item) lo = mid; else hi = mid;
    }
    return S.rows[lo];
}

// Is `pi` the first probe (table order, text length n = m + delta) whose segment equals the pattern's residues?
__device__ __noinline__ bool first_matching_probe(const JoinTables& tab, const uint32_t* __restrict__ prow,
                                                  const uint32_t* __restrict__ trow, int m, int n, int delta, int pi) {
    for (int k = 0; k <= pi; ++k) {
        const int i = tab.probe_seg[delta][k], d = tab.probe_shift[delta][k];
        const int sq = tab.seg_start[n][i], len = tab.seg_start[n][i + 1] - sq, rq = sq + d;
        if (rq < 0 || rq + len > m) continue;
        const bool eq = seg_equal(prow, rq, trow, sq, len);
        if (k == pi) return eq;
        if (eq) return false;
    }
    return false;
}

template <int R>
__device__ __forceinline__ void load_row(const uint32_t* __restrict__ row, uint32_t (&T)[R]) {
#pragma unroll
    for (int w = 0; w < R; w += 4) {
        const uint4 v = __ldg(reinterpret_cast<const uint4*>(row + w));
        T[w] = v.x, T[w + 1] = v.y, T[w + 2] = v.z, T[w + 3] = v.w;
    }
}

// residue j (a compile-time constant after unrolling) of a row held in registers
template <int R>
__device__ __forceinline__ uint32_t row_code(const uint32_t (&T)[R], int j) {
    const int pos = 5 * j, w = pos >> 5, sh = pos & 31;
    const uint32_t v = (sh <= 27 || w + 1 >= R) ? (T[w] >> sh) : __funnelshift_r(T[w], T[w + 1], sh);
    return v & 31u;
}

// ---- general kernel: candidates verified by the column recurrence ----
template <typename W>
__host__ __device__ constexpr int join_peq_row_bytes() {
    return 33 * (int)sizeof(W);
}
template <typename W>
__host__ __device__ constexpr int join_warp_smem_bytes() {
    return ((kPeqRows * join_peq_row_bytes<W>() + 15) & ~15) + kJoinQueue * 2 * 32 * 4;
}

template <typename W, int R, bool COUNT>
struct JoinWarp {
    uint32_t lane_addr;   // shared address of this lane's Peq column
    uint32_t queue_addr;  // shared address of this lane's candidate queue: [slot][text, probe] x 128 B
    const uint32_t* prow; // this lane's pattern row in seq5
    W pv_init;
    int lane, p, m, qn;
    bool p_valid;
    unsigned long long n_cols = 0, n_live = 0, n_tests = 0, n_cand = 0, n_probes = 0, n_entries = 0;
};

// Verify the queued candidates (texts of length n = m + delta), one per lane and round, in lock step.
template <typename W, int R, bool COUNT>
__device__ __forceinline__ void join_drain(JoinWarp<W, R, COUNT>& w, const JoinParams& S, int n, int delta) {
    constexpr int kCols = (32 * R) / 5 < kMaxLen ? (32 * R) / 5 : kMaxLen;
    constexpr int kRowBytes = join_peq_row_bytes<W>();
    const int l_max = S.d.l_max;
    while (__any_sync(kFullMask, w.qn > 0)) {
        const bool has = w.qn > 0;
        int t = w.p, pi = 0;
        if (has) {
            --w.qn;
            uint32_t a, b;
            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(a) : "r"(w.queue_addr + (uint32_t)w.qn * 256u));
            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(b) : "r"(w.queue_addr + (uint32_t)w.qn * 256u + 128u));
            t = (int)a, pi = (int)b;
        }
        const uint32_t* trow = S.seq5 + (size_t)t * S.s5_words;
        uint32_t T[R];
        load_row<R>(trow, T);
        W Pv = w.pv_init, Mv = W(0), bm = W(1);
        int dg = has ? delta : kJoinDead;  // D[0][delta] = delta: the first cell of the final diagonal
        if (COUNT) w.n_cand += (unsigned long long)__popc(__ballot_sync(kFullMask, has));
#pragma unroll
        for (int j = 0; j < kCols; ++j) {
            if (j >= n) break;  // warp-uniform
            if (COUNT) {
                w.n_cols += 32;
                w.n_live += (unsigned long long)__popc(__ballot_sync(kFullMask, dg <= l_max));
            }
            const W D0 = column_step<W>(peq_load<W, kRowBytes>(w.lane_addr, row_code<R>(T, j)), Pv, Mv);
            if (j >= delta) {  // row j + 1 - delta of the pattern exists: D[i][j+1] = D[i-1][j] + 1 - D0[bit i-1]
                if ((D0 & bm) == W(0)) ++dg;
                bm += bm;
                if (COUNT) w.n_tests += 32;
                if (!__any_sync(kFullMask, dg <= l_max)) break;
            }
        }
        bool edge = has && dg <= l_max;  // after column n, dg = D[m][n] = lev(pattern, text)
        if (edge) edge = first_matching_probe(S.tab, w.prow, trow, w.m, n, delta, pi);
        emit_edges(S.d, edge, w.lane, w.p, t, w.m, n);
    }
}

template <typename W, int R, bool COUNT>
__global__ void __launch_bounds__(kJoinThreads) k_join(const __grid_constant__ JoinParams S) {
    extern __shared__ __align__(16) unsigned char smem[];
    constexpr int kRowBytes = join_peq_row_bytes<W>();
    constexpr int kWarpBytes = join_warp_smem_bytes<W>();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned char* wsmem = smem + warp * kWarpBytes;
    W* peq = reinterpret_cast<W*>(wsmem);
    const uint32_t peq_addr = (uint32_t)__cvta_generic_to_shared(wsmem);

    JoinWarp<W, R, COUNT> w;
    w.lane = lane;
    w.lane_addr = peq_addr + lane * (uint32_t)sizeof(W);
    w.queue_addr = peq_addr + ((kPeqRows * kRowBytes + 15) & ~15) + lane * 4u;
    const DistanceParams& P = S.d;
    const int l_max = P.l_max;
    const long long n_local = (P.n_items - P.shard + P.n_shards - 1) / P.n_shards;
    for (;;) {
        unsigned long long q = 0;
        if (lane == 0) q = atomicAdd(P.queue, 1ull);
        q = __shfl_sync(kFullMask, q, 0);
        if ((long long)q >= n_local) break;
        const int64_t item = (int64_t)q * P.n_shards + P.shard;
        const JoinRow& Rw = find_join_row(S, item);
        const int m = Rw.m;
        const int p_rel = (int)(item - Rw.item_begin) * 32 + lane;
        w.p_valid = p_rel < Rw.p_count;
        w.p = Rw.p_start + (w.p_valid ? p_rel : 0);
        w.m = m;
        w.prow = S.seq5 + (size_t)w.p * S.s5_words;
        w.pv_init = low_mask<W>(m);
        w.qn = 0;
        __syncwarp();  // the previous item's Peq reads are done
        build_peq<W, kRowBytes>(peq, lane, w.p_valid, P.pat + (size_t)w.p * P.pat_stride, m);
        __syncwarp();

        for (int delta = 0; delta <= l_max; ++delta) {
            if (Rw.t_count[delta] == 0) continue;  // warp-uniform
            const int n = m + delta;
            const int np = S.tab.n_probes[delta];
            uint32_t e = 0, e_end = 0, tag = 0;
            int pi = -1;  // the probe being scanned
            for (bool last = false; !last;) {
                if (!__any_sync(kFullMask, e < e_end)) {
                    // every lane has walked its bucket: the next probe whose segment fits at its shift (warp-uniform)
                    int len = 0, rq = 0, i = 0;
                    for (++pi; pi < np; ++pi) {
                        i = S.tab.probe_seg[delta][pi];
                        const int sq = S.tab.seg_start[n][i];
                        len = S.tab.seg_start[n][i + 1] - sq;
                        rq = sq + S.tab.probe_shift[delta][pi];
                        if (rq >= 0 && rq + len <= m) break;
                    }
                    if (pi >= np) {
                        last = true;  // verify what is queued: the next delta has another text length
                    } else if (w.p_valid) {
                        const unsigned long long h = seg_hash(w.prow, rq, len, n, i);
                        const uint32_t b = (uint32_t)h & S.index.mask;
                        e = __ldg(S.index.dir + b);
                        e_end = __ldg(S.index.dir + b + 1);
                        tag = (uint32_t)(h >> 32);
                        if (COUNT) w.n_probes += (unsigned long long)__popc(__activemask());
                    }
                }
                if (e < e_end) {
                    const uint2 ent = __ldg(S.index.entries + e);
                    ++e;
                    if (COUNT) ++w.n_entries;
                    // same bucket: only the texts after the pattern (every unordered pair once)
                    if (ent.x == tag && (delta > 0 || (int)ent.y > w.p)) {
                        asm volatile("st.shared.u32 [%0], %1;" ::"r"(w.queue_addr + (uint32_t)w.qn * 256u), "r"(ent.y) : "memory");
                        asm volatile("st.shared.u32 [%0], %1;" ::"r"(w.queue_addr + (uint32_t)w.qn * 256u + 128u), "r"((uint32_t)pi) : "memory");
                        ++w.qn;
                    }
                }
                if (last || __any_sync(kFullMask, w.qn == kJoinQueue)) join_drain<W, R, COUNT>(w, S, n, delta);
            }
        }
    }
    if (COUNT) {
        // per-lane counters (entries) are summed over the warp; the others are warp-level already
        unsigned long long ne = w.n_entries;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) ne += __shfl_xor_sync(kFullMask, ne, o);
        if (lane == 0) {
            atomicAdd(P.work + 0, w.n_cols);
            atomicAdd(P.work + 1, w.n_tests);
            atomicAdd(P.work + 4, w.n_live);
            atomicAdd(P.work + 5, w.n_probes);
            atomicAdd(P.work + 6, ne);
            atomicAdd(P.work + 7, w.n_cand);
        }
    }
}

// ---- l_max <= 1 fast path: no recurrence at all ----
// all bits at positions >= pos of x are zero
template <int R>
__device__ __forceinline__ bool high_bits_zero(const uint32_t (&x)[R], int pos) {
    uint32_t acc = 0u;
#pragma unroll
    for (int w = 0; w < R; ++w) {
        const int lo = pos - 32 * w;
        acc |= lo <= 0 ? x[w] : (lo >= 32 ? 0u : (x[w] >> lo));
    }
    return acc == 0u;
}
template <int R>
__device__ __forceinline__ int first_set_bit(const uint32_t (&x)[R]) {  // -1: none
    int fb = -1;
#pragma unroll
    for (int w = R - 1; w >= 0; --w)
        if (x[w]) fb = 32 * w + __ffs((int)x[w]) - 1;
    return fb;
}
// lev(a, b) <= l_max for l_max <= 1, |b| = |a| + delta, delta in {0, 1}; rows are zero beyond the sequence.
//   equal lengths: the XOR of the packed codes is zero (identical) or confined to ONE 5-bit field (one substitution);
//   one longer:    with f = length of the common prefix, a[f..m) must equal b[f+1..m+1): b with residue f deleted.
template <int R>
__device__ __forceinline__ bool within_one(const uint32_t (&a)[R], const uint32_t (&b)[R], int m, int delta, int l_max) {
    uint32_t x[R];
#pragma unroll
    for (int w = 0; w < R; ++w) x[w] = a[w] ^ b[w];
    const int fb = first_set_bit<R>(x);
    if (delta == 0) {
        if (fb < 0) return true;
        if (l_max == 0) return false;
        const int f = fb / 5;
        return high_bits_zero<R>(x, 5 * f + 5);
    }
    const int f = fb < 0 ? m : min(fb / 5, m);
    uint32_t y[R];
#pragma unroll
    for (int w = 0; w < R; ++w) y[w] = a[w] ^ (w + 1 < R ? __funnelshift_r(b[w], b[w + 1], 5) : (b[w] >> 5));
    return high_bits_zero<R>(y, 5 * f);
}

template <int R, bool COUNT>
__global__ void __launch_bounds__(kJoinThreads) k_join_l1(const __grid_constant__ JoinParams S) {
    const int lane = threadIdx.x & 31;
    const DistanceParams& P = S.d;
    const int l_max = P.l_max;
    const long long n_local = (P.n_items - P.shard + P.n_shards - 1) / P.n_shards;
    unsigned long long n_cand = 0, n_probes = 0, n_entries = 0;
    for (;;) {
        unsigned long long q = 0;
        if (lane == 0) q = atomicAdd(P.queue, 1ull);
        q = __shfl_sync(kFullMask, q, 0);
        if ((long long)q >= n_local) break;
        const int64_t item = (int64_t)q * P.n_shards + P.shard;
        const JoinRow& Rw = find_join_row(S, item);
        const int m = Rw.m;
        const int p_rel = (int)(item - Rw.item_begin) * 32 + lane;
        const bool p_valid = p_rel < Rw.p_count;
        const int p = Rw.p_start + (p_valid ? p_rel : 0);
        const uint32_t* prow = S.seq5 + (size_t)p * S.s5_words;
        uint32_t A[R];
        load_row<R>(prow, A);
        for (int delta = 0; delta <= l_max; ++delta) {
            if (Rw.t_count[delta] == 0) continue;
            const int n = m + delta;
            const int np = S.tab.n_probes[delta];
            for (int pi = 0; pi < np; ++pi) {
                const int i = S.tab.probe_seg[delta][pi], d = S.tab.probe_shift[delta][pi];
                const int sq = S.tab.seg_start[n][i], len = S.tab.seg_start[n][i + 1] - sq, rq = sq + d;
                if (rq < 0 || rq + len > m) continue;
                uint32_t e = 0, e_end = 0, tag = 0;
                if (p_valid) {
                    const unsigned long long h = seg_hash(prow, rq, len, n, i);
                    const uint32_t b = (uint32_t)h & S.index.mask;
                    e = __ldg(S.index.dir + b);
                    e_end = __ldg(S.index.dir + b + 1);
                    tag = (uint32_t)(h >> 32);
                }
                if (COUNT) n_probes += (unsigned long long)__popc(__ballot_sync(kFullMask, p_valid));
                while (__any_sync(kFullMask, e < e_end)) {
                    bool edge = false;
                    int t = p;
                    if (e < e_end) {
                        const uint2 ent = __ldg(S.index.entries + e);
                        ++e;
                        if (COUNT) ++n_entries;
                        if (ent.x == tag && (delta > 0 || (int)ent.y > p)) {
                            t = (int)ent.y;
                            const uint32_t* trow = S.seq5 + (size_t)t * S.s5_words;
                            uint32_t B[R];
                            load_row<R>(trow, B);
                            if (COUNT) ++n_cand;
                            edge = within_one<R>(A, B, m, delta, l_max);
                            if (edge) edge = first_matching_probe(S.tab, prow, trow, m, n, delta, pi);
                        }
                    }
                    emit_edges(P, edge, lane, p, t, m, n);
                }
            }
        }
    }
    if (COUNT) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            n_entries += __shfl_xor_sync(kFullMask, n_entries, o);
            n_cand += __shfl_xor_sync(kFullMask, n_cand, o);
        }
        if (lane == 0) {
            atomicAdd(P.work + 5, n_probes);
            atomicAdd(P.work + 6, n_entries);
            atomicAdd(P.work + 7, n_cand);
        }
    }
}

template <typename K>
cudaError_t launch_persistent(K kern, const JoinParams& S, size_t smem, int ctas_per_sm, int n_sm, cudaStream_t s) {
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    const int64_t n_local = (S.d.n_items - S.d.shard + S.d.n_shards - 1) / S.d.n_shards;
    const int64_t ctas = std::max<int64_t>(1, std::min<int64_t>((int64_t)n_sm * ctas_per_sm, (n_local + kJoinWarps - 1) / kJoinWarps));
    kern<<<(unsigned)ctas, kJoinThreads, smem, s>>>(S);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_join_index(const uint32_t* seq5, int s5_words, const LengthTable& lt, int64_t n, const JoinTables& tab,
                              uint32_t* cnt, uint32_t* dir, uint2* entries, uint32_t slots, void* scan_scratch,
                              cudaStream_t s, int* launches) {
    const int64_t threads = n * tab.n_seg;
    if (threads <= 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((threads + 255) / 256);
    k_join_index<false><<<blocks, 256, 0, s>>>(seq5, s5_words, lt, n, tab, cnt, nullptr, nullptr, slots - 1u);
    *launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    e = exclusive_scan_u32_total(cnt, dir, (int64_t)slots, scan_scratch, s, launches);
    if (e != cudaSuccess) return e;
    k_join_index<true><<<blocks, 256, 0, s>>>(seq5, s5_words, lt, n, tab, cnt, dir, entries, slots - 1u);
    *launches += 1;
    return cudaGetLastError();
}

size_t join_smem_bytes(bool wide) {
    return (size_t)kJoinWarps * (wide ? join_warp_smem_bytes<uint64_t>() : join_warp_smem_bytes<uint32_t>());
}

cudaError_t launch_join(const DistanceParams& p, const JoinRow* rows, int n_rows, const uint32_t* seq5, int s5_words,
                        const JoinIndex& index, const JoinTables& tab, bool wide, bool fast_l1, bool count_work, int n_sm,
                        cudaStream_t s, int* launches) {
    if (p.n_items <= p.shard || n_rows <= 0) return cudaSuccess;
    JoinParams S{};
    S.d = p;
    S.rows = rows;
    S.n_rows = n_rows;
    S.s5_words = s5_words;
    S.seq5 = seq5;
    S.index = index;
    S.tab = tab;
    *launches += 1;
    if (fast_l1) {
        if (p.l_max > 1) return cudaErrorInvalidValue;
        // rows are read in full: patterns of <= 32 residues pair with texts of <= 33 (8 words are enough)
        const int r = wide ? s5_words : std::min(s5_words, 8);
        switch (r) {
            case 4: return count_work ? launch_persistent(k_join_l1<4, true>, S, 0, 8, n_sm, s) : launch_persistent(k_join_l1<4, false>, S, 0, 8, n_sm, s);
            case 8: return count_work ? launch_persistent(k_join_l1<8, true>, S, 0, 8, n_sm, s) : launch_persistent(k_join_l1<8, false>, S, 0, 8, n_sm, s);
            case 12: return count_work ? launch_persistent(k_join_l1<12, true>, S, 0, 8, n_sm, s) : launch_persistent(k_join_l1<12, false>, S, 0, 8, n_sm, s);
            default: return cudaErrorInvalidValue;
        }
    }
    const size_t smem = join_smem_bytes(wide);
    if (!wide) {
        // patterns of <= 32 residues: texts of <= 32 + l_max <= 36 residues = 180 bits: 8 words at most
        if (s5_words == 4)
            return count_work ? launch_persistent(k_join<uint32_t, 4, true>, S, smem, 4, n_sm, s)
                              : launch_persistent(k_join<uint32_t, 4, false>, S, smem, 4, n_sm, s);
        return count_work ? launch_persistent(k_join<uint32_t, 8, true>, S, smem, 4, n_sm, s)
                          : launch_persistent(k_join<uint32_t, 8, false>, S, smem, 4, n_sm, s);
    }
    if (s5_words == 8)
        return count_work ? launch_persistent(k_join<uint64_t, 8, true>, S, smem, 2, n_sm, s)
                          : launch_persistent(k_join<uint64_t, 8, false>, S, smem, 2, n_sm, s);
    if (s5_words == 12)
        return count_work ? launch_persistent(k_join<uint64_t, 12, true>, S, smem, 2, n_sm, s)
                          : launch_persistent(k_join<uint64_t, 12, false>, S, smem, 2, n_sm, s);
    return cudaErrorInvalidValue;
}

}  // namespace tcrnet

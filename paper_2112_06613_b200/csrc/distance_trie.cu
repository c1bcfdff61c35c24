// Steps A3-A5, prefix-trie kernel (the default whenever the early exit is on, l_max <= kTrieMaxL and
// the texts are longer than the trie is deep).
//
// Same arithmetic as distance.cu - the Myers/Hyyro column recurrence of myers.cuh, the exact
// final-diagonal early exit, warp-aggregated emission - but the texts of a
// length bucket are visited through the prefix trie of trie.cu instead of one by one:
//
//   * One work item = one warp = 32 patterns of one length (one per lane, neighbours in lexicographic
//     order, Peq column private in shared memory) against a chunk [lo, hi) of the sorted texts of one
//     length.  The kernel is persistent: every warp claims items from a device-wide queue until it is
//     empty.  The warp walks the trie depth-first.  Entering a level-k node
//     costs ONE column step (its residue code at position k-1) on top of the parent's (Pv, Mv):
//     the columns of a shared prefix are computed once per node, not once per text.
//   * The final-diagonal cell is TRACKED, not recomputed: with i = k - delta (delta = n - m),
//     dg = D[i][k] is carried along the walk and a column step updates it from its own D0 word,
//         D[i][k] = D[i-1][k-1] + 1 - D0[bit i-1]        (D0 bit = "the diagonal did not increase"),
//     starting from D[0][delta] = delta.  DP values never decrease along a diagonal and
//     lev(pattern, text) = D[m][n] is the last cell of this one, so dg > l_max in all 32 lanes kills
//     the node with its whole subtree ("abort, as soon as the smallest intermediate
//     result exceeds" l_max - here one abort disposes of a whole run of texts), and after the last
//     column dg IS the distance: no popcount anywhere.
//   * Dead children are not even visited ("guided expansion"; levels k <= l_max have no dead
//     children and are walked in full).  Before a node's children are walked, every lane derives
//     from its parent column (Pv, Mv, dg = D[i-1][k-1]) the exact set V of residue codes c whose
//     child would be alive, i.e. D_c[i][k] = dg + 1 - D0_c[bit i-1] <= l_max:
//         dg <  l_max                       V = all codes
//         dg == l_max, Mv[bit i-1] set      V = all codes      (D0_c >= Mv for every c)
//         dg == l_max                       V = { a_i } + { a_(i-t) : Pv[bits i-1-t .. i-2] all set, t >= 1 }
//         dg >  l_max                       V = {}             (the lane is dead for good)
//     (the three terms of D0 = carry | Eq | Mv; a carry reaches bit i-1 from a match at bit i-1-t
//     through t set bits of Pv).  D[i-1-t][k-1] = dg - t >= delta + t bounds t by (l_max - delta) / 2,
//     so the t-loop has 0 iterations for l_max <= 1, one for l_max <= 3, two for l_max = 4.
//     The warp visits the children whose code is in the OR of the 32 lanes' V (one REDUX) and in the
//     node's child-code bitmap.  V is exact, so no per-child test is needed.
//   * Texts below a surviving level-kTrieDepth node are finished column by column from the node's
//     state (a vote after every second column); surviving pairs (dg <= l_max after column n) are
//     emitted as in distance.cu.
//
// Everything a warp does is warp-uniform (all lanes visit the same node / text), so there is no
// divergence; lanes differ only in their pattern.  The children of the node being expanded
// (<= 27, plus the next node as sentinel) are fetched with one coalesced 128-bit load per lane and
// staged in a per-warp, per-level shared-memory buffer INDEXED BY RESIDUE CODE as
// (text_begin, text_end, child_begin, child_codes); the walk reads a child with one broadcast LDS.128.
//
// The kernel is specialised on l_max (template LMAX = 0..kTrieMaxL): thresholds are immediates and
// the t-loop is unrolled to its exact trip count.  delta is run-time but warp-uniform; it enters only
// through six precomputed bit masks.
#include <algorithm>

#include "myers.cuh"

namespace tcrnet {
namespace {

constexpr uint32_t kFull = 0xffffffffu;
constexpr int kTrieWarps = 8;                    // warps per CTA (independent of each other)
constexpr int kTrieThreads = 32 * kTrieWarps;
// Per-warp shared memory: Peq[kPeqRows][kTrieTile + 1 words] (the odd row stride keeps the row address a true
// multiply-add, which ptxas issues on the FMA pipe), then the staging buffers [kTrieDepth][kTrieFan] x 16 B.
template <typename W>
__host__ __device__ constexpr int trie_peq_row_bytes() {
    return (kTrieTile + 1) * (int)sizeof(W);
}
template <typename W>
__host__ __device__ constexpr int trie_warp_smem_bytes() {
    return ((kPeqRows * trie_peq_row_bytes<W>() + 15) & ~15) + kTrieDepth * kTrieFan * 16 + kTrieDepth * 128;
}
constexpr int kClipLevels = 3;      // levels whose nodes are clipped to the work item's text chunk
constexpr int kDeadLane = 1 << 20;  // dg of a lane without a pattern: never alive, never emitted

template <typename W, bool COUNT>
struct Walk {
    uint32_t stage_addr;      // shared address of this warp's staging buffers: [kTrieDepth][kTrieFan] children by code
    uint32_t lane_addr;       // shared address of this lane's Peq column
    const uint32_t* rows;     // text row of sorted position 0 of this bucket's numbering (bucket base - t_start rows)
    uint32_t lo, hi;          // texts [lo, hi) (sorted positions) are this warp's share of the bucket
    uint32_t ohs_addr;        // shared address of this lane's one-hot codes: [q - 1] = 1 << code of pattern row q - delta
                              // (0: no such row / no pattern), q = 1..kTrieDepth, stride 128 B
    uint32_t dsh;             // delta + 1: the bit of pattern row q - delta is (1 << q) >> dsh (0 when q <= delta)
    W pv_init;
    int rw, n;
    int lane, p_sorted;
    int p_lim;                // same bucket: p_sorted (only sorted p < t counts); else -1
    unsigned long long n_cols = 0, n_tests = 0, n_first = 0, n_vsets = 0;

    __device__ __forceinline__ uint32_t dbit(int q) const { return (1u << q) >> dsh; }
};

__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts32(uint32_t addr, uint32_t v) {
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void sts128(uint32_t addr, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
// Pin a value in a register: the compiler may not recompute it from its definition (threadIdx, the shared window).
__device__ __forceinline__ void keep(uint32_t& x) { asm volatile("" : "+r"(x)); }

// Columns j0 + Q0 .. j0 + 3 of one text (residue codes c4; FULL: all of them exist, else only those < n).
// Returns false when the exit vote kills the text (dg > l_max in all 32 lanes).
template <typename W, int LMAX, bool COUNT, int Q0, bool FULL>
__device__ __forceinline__ bool columns4(Walk<W, COUNT>& w, const uint4 c4, int j0, W& Pv, W& Mv, W& bm, int& dg) {
    // exit vote after every column, or after every second one for l_max <= 1 (measured: cfg4 / cfg5)
    constexpr int kVoteEvery = LMAX >= 2 ? 1 : 2;
    const uint32_t c[4] = {c4.x, c4.y, c4.z, c4.w};
#pragma unroll
    for (int q = Q0; q < 4; ++q) {
        if (!FULL && j0 + q >= w.n) return true;  // warp-uniform
        const W D0 = column_step<W>(peq_load<W, trie_peq_row_bytes<W>()>(w.lane_addr, c[q]), Pv, Mv);
        if ((D0 & bm) == W(0)) ++dg;
        bm += bm;
        if (COUNT) ++w.n_cols;
        if (kVoteEvery == 1 || (q & 1)) {
            if (COUNT) ++w.n_tests;
            if (!__any_sync(kFull, dg <= LMAX)) return false;
        }
    }
    return true;
}

// The texts [t0, t1) below a surviving deepest-level node, one by one: the text columns kTrieDepth .. n-1
// (0-based) on top of the node's state (Pv0, Mv0, dg0) with the tracked final-diagonal cell; emission.
// (Leaving the trie earlier for subtrees of one or two texts was measured and is slower: the walk's exact
// V sets prune more than the votes of this loop.)
template <typename W, int LMAX, bool COUNT>
__device__ __forceinline__ void finish_texts(Walk<W, COUNT>& w, const DistanceParams& P, uint32_t t0, uint32_t t1,
                                             uint4 c4, const W Pv0, const W Mv0, const int dg0) {
    constexpr int START = kTrieDepth;
    static_assert(START >= 1 && START >= kTrieMaxL, "column 0 has its own step; final-diagonal rows exist from column delta on");
    constexpr int kJ0 = START & ~3;  // the 128-bit load that holds column START
    // c4 = the first columns of text t0 (requested by the caller before its own column step); those of text t + 1
    // are requested before text t is processed, so the L2 latency of a row overlaps the previous text's columns
    for (uint32_t t = t0; t < t1; ++t) {
        const uint4* row = reinterpret_cast<const uint4*>(w.rows + (size_t)t * w.rw);
        const uint4 c4_here = c4;
        if (t + 1u < t1) c4 = __ldg(row + ((w.rw + kJ0) >> 2));
        W Pv = Pv0, Mv = Mv0;
        W bm = (W)w.dbit(START + 1);  // bit of row j + 1 - delta for column j = START
        int dg = dg0;
        // four columns per 128-bit load (the same address in all lanes)
        int j0 = kJ0;
        bool alive;
        {
            alive = kJ0 + 4 <= w.n ? columns4<W, LMAX, COUNT, START & 3, true>(w, c4_here, kJ0, Pv, Mv, bm, dg)
                                   : columns4<W, LMAX, COUNT, START & 3, false>(w, c4_here, kJ0, Pv, Mv, bm, dg);
            j0 += 4;
        }
        while (alive && j0 + 4 <= w.n) {
            alive = columns4<W, LMAX, COUNT, 0, true>(w, __ldg(row + (j0 >> 2)), j0, Pv, Mv, bm, dg);
            j0 += 4;
        }
        if (alive && j0 < w.n) alive = columns4<W, LMAX, COUNT, 0, false>(w, __ldg(row + (j0 >> 2)), j0, Pv, Mv, bm, dg);
        if (!alive) continue;
        const bool edge = dg <= LMAX && w.p_lim < (int)t;
        emit_edges(P, edge, w.lane, w.p_sorted, (int)t, w.n - (int)w.dsh + 1, w.n);
    }
}

// Lane i's share of the children [cb, cb + popc(cm)] of a node (the last one is the next node or the sentinel).
template <int LEVEL>
__device__ __forceinline__ uint4 load_children(const DistanceParams& P, uint32_t cb, uint32_t cm, int lane) {
    return __ldg(reinterpret_cast<const uint4*>(P.trie[LEVEL]) + (cb + min((uint32_t)lane, (uint32_t)__popc(cm))));
}

// Expand the children (level LEVEL, nodes [cb, cb + popc(cm)), residue codes = the set bits of cm) of
// one level-(LEVEL-1) node, or the roots of the text bucket.  (Pv, Mv) is the DP column after LEVEL-1
// text residues and dg = D[LEVEL-1-delta][LEVEL-1] its final-diagonal cell (delta while there is none).
template <typename W, int LMAX, bool COUNT, int LEVEL>
__device__ __forceinline__ void visit(Walk<W, COUNT>& w, const DistanceParams& P, uint32_t cm, const uint4 nd_lane,
                                      const W Pv, const W Mv, const int dg) {
    uint32_t U = cm;
    // Guided expansion: the codes whose child is alive in at least one lane.  Every child is alive
    // while LEVEL <= l_max (D[i][k] <= k); LEVEL > l_max >= delta, so row i = LEVEL - delta exists.
    if constexpr (LEVEL > LMAX) {
        const uint32_t b = w.dbit(LEVEL);
        uint32_t V = lds32(w.ohs_addr + (LEVEL - 1) * 128);
#pragma unroll
        for (int t = 1; t <= LMAX / 2; ++t) {
            const uint32_t run = b - (b >> t);  // bits i-1-t .. i-2 (b itself when there is no row i-t: ohs = 0)
            if (((uint32_t)Pv & run) == run) V |= lds32(w.ohs_addr + (LEVEL - t - 1) * 128);
        }
        if (dg != LMAX) V = 0u;
        if (dg < LMAX || (dg == LMAX && ((uint32_t)Mv & b) != 0u)) V = kFull;
        if (COUNT) ++w.n_vsets;
        U = __reduce_or_sync(kFull, V) & cm;
        if (U == 0u) return;
    }
    const uint32_t sb = w.stage_addr + (LEVEL - 1) * kTrieFan * 16;
    {
        const uint32_t cnt = (uint32_t)__popc(cm);  // <= 27 by construction; node cb + cnt is the next node or the sentinel
        __syncwarp();
        const uint4 nd = nd_lane;  // child min(lane, cnt), requested by the caller before its own column step
        const uint32_t text_end = __shfl_down_sync(kFull, nd.x, 1);
        if ((uint32_t)w.lane < cnt) sts128(sb + nd.z * 16, nd.x, text_end, nd.y, nd.w);  // code < kTrieFan
        __syncwarp();
    }
    do {
        const uint32_t c = (uint32_t)__ffs((int)U) - 1u;  // children in ascending code order
        U &= U - 1u;
        const uint4 nd = lds128(sb + c * 16);  // text_begin, text_end, child_begin, child_codes
        if (LEVEL <= kClipLevels) {  // clip the upper levels to this warp's texts
            if (nd.y <= w.lo || nd.x >= w.hi) continue;
        }
        // what the walk needs below this child - its children (one per lane), or the first columns of its first
        // text - is requested now: the L2 latency overlaps the column step and the V sets
        uint4 below = make_uint4(0u, 0u, 0u, 0u);
        uint32_t t0 = 0u, t1 = 0u;
        if constexpr (LEVEL < kTrieDepth) {
            below = load_children<LEVEL + 1>(P, nd.z, nd.w, w.lane);
        } else {
            t0 = max(nd.x, w.lo), t1 = min(nd.y, w.hi);
            if (t0 >= t1) continue;
            below = __ldg(reinterpret_cast<const uint4*>(w.rows + (size_t)t0 * w.rw) + (kTrieDepth >> 2));
        }
        const W Eq = peq_load<W, trie_peq_row_bytes<W>()>(w.lane_addr, c);
        W P2 = Pv, M2 = Mv;
        W D0;
        if (LEVEL == 1) {
            D0 = first_column_step<W>(Eq, w.pv_init, w.pv_init + w.pv_init, P2, M2);
            if (COUNT) ++w.n_first;
        } else {
            D0 = column_step<W>(Eq, P2, M2);
        }
        if (COUNT) ++w.n_cols;
        int dg2 = dg;
        if (LEVEL > LMAX || LEVEL >= (int)w.dsh) {  // row LEVEL - delta >= 1 exists (warp-uniform)
            if (((uint32_t)D0 & w.dbit(LEVEL)) == 0u) ++dg2;
        }
        if constexpr (LEVEL < kTrieDepth) {
            visit<W, LMAX, COUNT, LEVEL + 1>(w, P, nd.w, below, P2, M2, dg2);
        } else {
            finish_texts<W, LMAX, COUNT>(w, P, t0, t1, below, P2, M2, dg2);
        }
    } while (U);
}

// One warp = one work item at a time: kTrieTile patterns of one length (neighbours in lexicographic order) against
// a chunk of one text bucket.  Items are claimed from a device-wide queue (one atomicAdd per item, big rows first),
// so a warp slot is never idle while work is left; each warp owns a private Peq table and staging buffer in shared
// memory and there is no CTA-level barrier anywhere.
template <typename W, int LMAX, bool COUNT>
__global__ void __launch_bounds__(kTrieThreads, sizeof(W) == 4 ? 4 : 2) k_distance_trie(const __grid_constant__ DistanceParams P) {
    extern __shared__ __align__(16) unsigned char smem[];
    constexpr int kRowBytes = trie_peq_row_bytes<W>();
    constexpr int kWarpBytes = trie_warp_smem_bytes<W>();

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned char* wsmem = smem + warp * kWarpBytes;
    W* peq = reinterpret_cast<W*>(wsmem);
    const uint32_t peq_addr = (uint32_t)__cvta_generic_to_shared(wsmem);

    Walk<W, COUNT> w;
    w.stage_addr = peq_addr + ((kPeqRows * kRowBytes + 15) & ~15);
    w.lane_addr = peq_addr + lane * (uint32_t)sizeof(W);
    w.ohs_addr = w.stage_addr + kTrieDepth * kTrieFan * 16 + lane * 4u;
    keep(w.stage_addr);
    keep(w.lane_addr);
    keep(w.ohs_addr);
    w.lane = lane;
    {
        uint32_t l = (uint32_t)w.lane;
        keep(l);
        w.lane = (int)l;
    }

    const long long n_local = (P.n_items - P.shard + P.n_shards - 1) / P.n_shards;  // step 8(e): interleaved shards
    for (;;) {
        // ---- step A2, device side: claim the next (bucket pair, pattern tile, text chunk) ----
        unsigned long long q = 0;
        if (lane == 0) q = atomicAdd(P.queue, 1ull);
        q = __shfl_sync(kFull, q, 0);
        if ((long long)q >= n_local) break;
        const int64_t item = (int64_t)q * P.n_shards + P.shard;
        const WorkRow R = find_row(P, item);
        const int64_t local = item - R.item_begin;
        const int pi = (int)(local / R.n_tchunks), qi = (int)(local % R.n_tchunks);
        const int p_tile0 = pi * kTrieTile;       // relative to the pattern bucket
        const int chunk_t0 = qi * R.tchunk;       // relative to the text bucket
        const int chunk_cnt = min(R.tchunk, R.t_count - chunk_t0);
        // same bucket: a warp pairs only with the texts after its first pattern (sorted p < t)
        const int lo_rel = R.diag ? max(chunk_t0, p_tile0 + 1) : chunk_t0;
        const int hi_rel = chunk_t0 + chunk_cnt;
        if (lo_rel >= hi_rel) continue;  // wholly on/below the diagonal

        const int m = R.m, n = R.n;
        const int delta = n - m;                  // 0 <= delta <= l_max = LMAX
        const int p_rel = p_tile0 + lane;
        const bool p_valid = p_rel < R.p_count;
        const uint8_t* prow = P.pat + (size_t)(R.p_start + p_rel) * P.pat_stride;
        __syncwarp();  // the previous item's Peq reads are done
        build_peq<W, kRowBytes>(peq, lane, p_valid, prow, m);

        w.rows = P.txt + R.txt_base - (size_t)R.t_start * R.row_words;
        w.lo = (uint32_t)(R.t_start + lo_rel);
        w.hi = (uint32_t)(R.t_start + hi_rel);
        w.dsh = (uint32_t)delta + 1u;
        keep(w.dsh);
        {
            // one-hot codes of the pattern's first rows, shifted by delta: ohs[q] belongs to row q - delta
            const uint2 head = p_valid ? __ldg(reinterpret_cast<const uint2*>(prow)) : make_uint2(0xffffffffu, 0xffffffffu);
#pragma unroll
            for (int k = 0; k <= kTrieDepth; ++k) {
                const int r = k - delta;  // 1-based pattern row
                uint32_t code = 0xffu;
                if (r >= 1 && r <= m) code = ((r <= 4 ? head.x : head.y) >> (8 * ((r - 1) & 3))) & 0xffu;
                if (k >= 1) sts32(w.ohs_addr + (k - 1) * 128, code < 32u ? 1u << code : 0u);
            }
        }
        w.pv_init = low_mask<W>(m);
        w.rw = R.row_words;
        w.n = n;
        w.p_sorted = R.p_start + p_rel;
        w.p_lim = R.diag ? w.p_sorted : -1;

        // codes of the bucket's level-1 nodes
        uint32_t root_codes = 0u;
        {
            const int cnt = (int)(R.root_end - R.root_begin);
            if (lane < cnt) root_codes = 1u << (P.trie[1][R.root_begin + lane].code & 31u);
            root_codes = __reduce_or_sync(kFull, root_codes);
        }
        // D[0][delta] = delta is the first cell of the final diagonal
        visit<W, LMAX, COUNT, 1>(w, P, root_codes, load_children<1>(P, R.root_begin, root_codes, lane), w.pv_init, W(0),
                                 p_valid ? delta : kDeadLane);
    }

    if (COUNT) {
        // warp-level counters (identical in all lanes): lane 0 reports 32 lanes' worth
        if (lane == 0) {
            atomicAdd(P.work + 0, w.n_cols * 32ull);
            atomicAdd(P.work + 1, w.n_tests * 32ull);
            atomicAdd(P.work + 2, w.n_first * 32ull);
            atomicAdd(P.work + 3, w.n_vsets * 32ull);
        }
    }
}

template <typename W, int LMAX, bool COUNT>
cudaError_t launch_one(const DistanceParams& p, int64_t n_items, size_t smem, int n_sm, cudaStream_t s) {
    auto kern = k_distance_trie<W, LMAX, COUNT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    // persistent: every warp slot the kernel can hold, or one warp per item if there are fewer
    const int64_t n_local = (n_items - p.shard + p.n_shards - 1) / p.n_shards;
    const int64_t ctas_full = (int64_t)n_sm * (sizeof(W) == 4 ? 4 : 2);
    const int64_t ctas = std::max<int64_t>(1, std::min(ctas_full, (n_local + kTrieWarps - 1) / kTrieWarps));
    kern<<<(unsigned)ctas, kTrieThreads, smem, s>>>(p);
    return cudaGetLastError();
}

template <typename W, int LMAX>
cudaError_t launch_lmax(const DistanceParams& p, int64_t n_items, bool count_work, size_t smem, int n_sm, cudaStream_t s) {
    return count_work ? launch_one<W, LMAX, true>(p, n_items, smem, n_sm, s)
                      : launch_one<W, LMAX, false>(p, n_items, smem, n_sm, s);
}

template <typename W>
cudaError_t launch_word(const DistanceParams& p, int64_t n_items, bool count_work, size_t smem, int n_sm, cudaStream_t s) {
    static_assert(kTrieMaxL == 4, "one case per specialised l_max");
    switch (p.l_max) {
        case 0: return launch_lmax<W, 0>(p, n_items, count_work, smem, n_sm, s);
        case 1: return launch_lmax<W, 1>(p, n_items, count_work, smem, n_sm, s);
        case 2: return launch_lmax<W, 2>(p, n_items, count_work, smem, n_sm, s);
        case 3: return launch_lmax<W, 3>(p, n_items, count_work, smem, n_sm, s);
        case 4: return launch_lmax<W, 4>(p, n_items, count_work, smem, n_sm, s);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

size_t distance_trie_smem_bytes(bool wide) {
    return (size_t)kTrieWarps * (wide ? trie_warp_smem_bytes<uint64_t>() : trie_warp_smem_bytes<uint32_t>());
}

cudaError_t launch_distance_trie(const DistanceParams& p, int64_t n_items, bool wide, bool count_work, int n_sm,
                                 cudaStream_t s, int* launches) {
    if (n_items <= p.shard) return cudaSuccess;
    const size_t smem = distance_trie_smem_bytes(wide);
    *launches += 1;
    return wide ? launch_word<uint64_t>(p, n_items, count_work, smem, n_sm, s)
                : launch_word<uint32_t>(p, n_items, count_work, smem, n_sm, s);
}

}  // namespace tcrnet

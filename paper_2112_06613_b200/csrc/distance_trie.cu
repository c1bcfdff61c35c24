// Steps A3-A5, prefix-trie kernel (the default whenever the early exit is on and can act within
// the first kTrieDepth text columns).
//
// Same arithmetic as distance.cu - the Myers/Hyyro column recurrence of myers.cuh, the exact
// final-diagonal early exit, warp-aggregated emission - but the texts of a
// length bucket are visited through the prefix trie of trie.cu instead of one by one:
//
//   * One CTA = 256 patterns of one length (one per thread, Peq column private in shared memory)
//     against a chunk [lo, hi) of the sorted texts of one length.  A warp (32 patterns that are
//     neighbours in lexicographic order) walks the trie depth-first.  Entering a level-k node
//     costs ONE column step (its residue code at position k-1) on top of the parent's (Pv, Mv):
//     the columns of a shared prefix are computed once per node, not once per text.
//   * Early exit: the cell D[k - delta][k] of the final diagonal is a lower bound of
//     lev(pattern, text) for EVERY text below a level-k node, so a node where it exceeds l_max in
//     all 32 lanes is dead with its whole subtree.  PAPER.md:326 ("abort, as soon as the smallest
//     intermediate result exceeds" l_max) - here one abort disposes of a whole run of texts.
//   * Dead children are not even visited ("guided expansion"; levels k <= l_max have no dead
//     children and are walked in full): before a node's children are walked, every lane derives from
//     its parent column (Pv, Mv) the exact set V of residue codes c whose child would be alive,
//         D_c[i][k] = min( D_0[i][k],  min over rows r <= i with a_r = c of D[r-1][k-1] + (i - r) ),
//     (i = k - delta; D_0 = the column of a code that matches nowhere), i.e.
//         V = (all codes, if D_0[i][k] <= l_max)  |  { a_(i-t) : D[i-1-t][k-1] + 2t <= l_max, t = 0..l_max }
//     with D_0[i][k] <= l_max  <=>  D[i][k-1] <= l_max - 1  or  D[i-1-u][k-1] <= l_max - 1 - 2u for
//     some u in 0..l_max-1.  Each cell costs one LOP3 + POPC + compare.  The warp visits the
//     children whose code is in the OR of the 32 lanes' V (one REDUX) and in the node's child-code
//     bitmap; the child's slot is popc(bitmap & low(code)).  V is exact, so no per-child test is
//     needed.
//   * Texts below a surviving level-kTrieDepth node are finished column by column from the node's
//     state (a test after every second column), then the distance is read off Pv / Mv and
//     surviving pairs are emitted as in distance.cu.
//
// Everything a warp does is warp-uniform (all lanes visit the same node / text), so there is no
// divergence; lanes differ only in their pattern.  The children of the node being expanded
// (<= 27, plus the next node as sentinel) are fetched with one coalesced 128-bit load per lane and
// staged in a per-warp, per-level shared-memory buffer; the walk then reads them with broadcast
// LDS.128.
//
// A cell needs one POPC: with v = ((Pv & 0xffff) | (Mv << 16)) ^ 0xffff0000 (PRMT + LOP3, once per
// node) and mask2(r) = low(r) in both halves, popc(v & mask2(r)) = popc(Pv & low(r)) + r - popc(Mv & low(r))
// = D[r][k-1] - (k-1) + r, so for r = i-1-u:  D[r][k-1] = popc(v & mask2(r)) + delta + u.
#include "myers.cuh"

namespace tcrnet {
namespace {

constexpr uint32_t kFull = 0xffffffffu;
constexpr int kClipLevels = 3;  // levels whose nodes are clipped to the work item's text chunk

template <typename W, bool COUNT>
struct Walk {
    uint4* stage;             // this warp's staging buffers: [kTrieDepth][kTrieFan] nodes
    const uint32_t* rows;     // first text row of the text bucket
    uint32_t lane_addr;       // shared address of this lane's Peq column
    uint32_t t_start;         // sorted position of the bucket's first text
    uint32_t lo, hi;          // texts [lo, hi) (sorted positions) are this warp's share of the bucket
    uint32_t mask2[kTrieDepth + 1];  // [q] = low(q - delta) in both 16-bit halves (0 when q <= delta)
    uint32_t ohs[kTrieDepth + 1];    // [q] = 1 << code of pattern row q - delta (0: no such row / no pattern)
    W pv_init, x_init, m_mask;
    int rw, n, delta;
    int thr;                  // l_max - delta; -1 in lanes without a pattern
    int l_max;                // warp-uniform
    int l_max_lane;           // l_max; -1 in lanes without a pattern
    int lane, p_sorted, diag;
    unsigned long long n_cols = 0, n_tests = 0, n_first = 0, n_ptests = 0;
};

// The texts [t0, t1) below a surviving deepest-level node: remaining columns, distance, emission.
template <typename W, bool COUNT>
__device__ __forceinline__ void finish_texts(Walk<W, COUNT>& w, const DistanceParams& P, uint32_t t0, uint32_t t1,
                                             const W Pv0, const W Mv0) {
    for (uint32_t t = t0; t < t1; ++t) {
        const uint32_t* row = w.rows + (size_t)(t - w.t_start) * w.rw;
        W Pv = Pv0, Mv = Mv0;
        bool dead = false;
        for (int j0 = kTrieDepth & ~3; j0 < w.n && !dead; j0 += 4) {
            const uint4 c4 = __ldg(reinterpret_cast<const uint4*>(row + j0));  // same address in all lanes
            const uint32_t c[4] = {c4.x, c4.y, c4.z, c4.w};
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int j = j0 + q;
                if (j < kTrieDepth || j >= w.n || dead) continue;
                column_step<W>(peq_load<W>(w.lane_addr, c[q]), Pv, Mv);
                if (COUNT) ++w.n_cols;
                const int jj = j + 1;
                if ((jj & 1) == 0 && jj < w.n && jj > w.delta) {
                    const W msk = low_mask<W>(jj - w.delta);
                    const int lb = jj + WordOps<W>::popc(Pv & msk) - WordOps<W>::popc(Mv & msk);
                    if (COUNT) ++w.n_tests;
                    if (!__any_sync(kFull, lb <= w.l_max_lane)) dead = true;
                }
            }
        }
        if (dead) continue;
        const int d = w.n + WordOps<W>::popc(Pv & w.m_mask) - WordOps<W>::popc(Mv & w.m_mask);
        const bool edge = d <= w.l_max_lane && (!w.diag || (uint32_t)w.p_sorted < t);
        emit_edges(P, edge, w.lane, w.p_sorted, (int)t, w.n - w.delta, w.n);
    }
}

// Expand the level-LEVEL nodes [cb, ce) (the children of one level-(LEVEL-1) node, or the roots of
// the text bucket) whose residue codes are the set bits of cm; (Pv, Mv) is the DP column after
// LEVEL-1 text residues.
template <typename W, bool COUNT, int LEVEL>
__device__ __forceinline__ void visit(Walk<W, COUNT>& w, const DistanceParams& P, uint32_t cb, uint32_t ce,
                                      uint32_t cm, const W Pv, const W Mv) {
    uint32_t U = cm;
    // Guided expansion: the codes whose child is alive in at least one lane.  Every child is alive
    // while LEVEL <= l_max (D[i][k] <= k), and there is no final-diagonal cell while LEVEL <= delta.
    if (LEVEL > w.l_max && LEVEL > w.delta) {  // warp-uniform
        const uint32_t v = __byte_perm((uint32_t)Pv, (uint32_t)Mv, 0x5410) ^ 0xffff0000u;
        bool alive0 = __popc(v & w.mask2[LEVEL]) <= w.thr;  // D[i][k-1] <= l_max - 1
        uint32_t V = 0u;
#pragma unroll
        for (int t = 0; t < LEVEL; ++t) {
            if (t <= w.l_max) {  // warp-uniform
                const int pt = __popc(v & w.mask2[LEVEL - 1 - t]);  // D[i-1-t][k-1] - delta - t
                alive0 = alive0 || (pt <= w.thr - 1 - 2 * t);
                if (pt <= w.thr - 2 * t) V |= w.ohs[LEVEL - t];
                if (COUNT) ++w.n_ptests;
            }
        }
        if (COUNT) ++w.n_ptests;
        if (alive0) V = kFull;
        U = __reduce_or_sync(kFull, V) & cm;
        if (U == 0u) return;
    }
    uint4* sb = w.stage + (LEVEL - 1) * kTrieFan;
    const int cnt = (int)(ce - cb);  // <= 27 by construction
    __syncwarp();
    if (w.lane <= cnt) sb[w.lane] = __ldg(reinterpret_cast<const uint4*>(P.trie[LEVEL]) + cb + w.lane);
    __syncwarp();
    do {
        const uint32_t c = (uint32_t)__ffs((int)U) - 1u;
        U &= U - 1u;
        const int i = __popc(cm & ((1u << c) - 1u));
        const uint4 nd = sb[i];      // text_begin, child_begin, code (= c), child codes
        const uint4 nx = sb[i + 1];
        if (LEVEL <= kClipLevels) {  // clip the upper levels to this warp's texts
            if (nx.x <= w.lo || nd.x >= w.hi) continue;
        }
        const W Eq = peq_load<W>(w.lane_addr, c);
        W P2 = Pv, M2 = Mv;
        if (LEVEL == 1) {
            first_column_step<W>(Eq, w.pv_init, w.x_init, P2, M2);
            if (COUNT) ++w.n_first;
        } else {
            column_step<W>(Eq, P2, M2);
        }
        if (COUNT) ++w.n_cols;
        if constexpr (LEVEL < kTrieDepth) {
            visit<W, COUNT, LEVEL + 1>(w, P, nd.y, nx.y, nd.w, P2, M2);
        } else {
            const uint32_t t0 = max(nd.x, w.lo), t1 = min(nx.x, w.hi);
            if (t0 < t1) finish_texts<W, COUNT>(w, P, t0, t1, P2, M2);
        }
    } while (U);
}

template <typename W, bool COUNT>
__global__ void __launch_bounds__(kTQ) k_distance_trie(const __grid_constant__ DistanceParams P) {
    extern __shared__ __align__(16) unsigned char smem[];
    constexpr int kRowBytes = peq_row_bytes<W>();
    static_assert((kPeqRows * kRowBytes) % 16 == 0, "the staging buffers follow the Peq table");
    W* peq = reinterpret_cast<W*>(smem);
    uint4* stage_all = reinterpret_cast<uint4*>(smem + kPeqRows * kRowBytes);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // ---- step A2, device side: which (bucket pair, pattern tile, text chunk) is this CTA? ----
    const int64_t item = work_item(P);
    const WorkRow R = find_row(P, item);
    const int64_t local = item - R.item_begin;
    const int pi = (int)(local / R.n_tchunks), qi = (int)(local % R.n_tchunks);
    const int p_tile0 = pi * kTQ;             // relative to the pattern bucket
    const int chunk_t0 = qi * R.tchunk;       // relative to the text bucket
    const int chunk_cnt = min(R.tchunk, R.t_count - chunk_t0);
    if (R.diag && chunk_t0 + chunk_cnt <= p_tile0 + 1) return;  // wholly on/below the diagonal

    const int m = R.m, n = R.n;
    const int delta = n - m;                  // 0 <= delta <= l_max
    const int p_rel = p_tile0 + tid;
    const bool p_valid = p_rel < R.p_count;
    build_peq<W>(peq, tid, p_valid, P.pat + (size_t)(R.p_start + p_rel) * P.pat_stride, m);

    // same bucket: a warp pairs only with the texts after its first pattern (sorted p < t)
    const int warp_p0 = p_tile0 + warp * 32;
    const int lo_rel = R.diag ? max(chunk_t0, warp_p0 + 1) : chunk_t0;
    const int hi_rel = chunk_t0 + chunk_cnt;
    if (lo_rel >= hi_rel || warp_p0 >= R.p_count) return;  // warp-uniform; no CTA barrier follows

    Walk<W, COUNT> w;
    w.stage = stage_all + warp * (kTrieDepth * kTrieFan);
    w.rows = P.txt + R.txt_base;
    w.lane_addr = (uint32_t)__cvta_generic_to_shared(smem) + tid * (uint32_t)sizeof(W);
    w.t_start = (uint32_t)R.t_start;
    w.lo = (uint32_t)(R.t_start + lo_rel);
    w.hi = (uint32_t)(R.t_start + hi_rel);
#pragma unroll
    for (int k = 0; k <= kTrieDepth; ++k) w.mask2[k] = k > delta ? ((1u << (k - delta)) - 1u) * 0x10001u : 0u;
    {
        // one-hot codes of the pattern's first rows, shifted by delta: ohs[q] belongs to row q - delta
        const uint8_t* prow = P.pat + (size_t)(R.p_start + p_rel) * P.pat_stride;
        const uint2 head = p_valid ? __ldg(reinterpret_cast<const uint2*>(prow)) : make_uint2(0xffffffffu, 0xffffffffu);
#pragma unroll
        for (int q = 0; q <= kTrieDepth; ++q) {
            const int r = q - delta;  // 1-based pattern row
            uint32_t code = 0xffu;
            if (r >= 1 && r <= m) code = ((r <= 4 ? head.x : head.y) >> (8 * ((r - 1) & 3))) & 0xffu;
            w.ohs[q] = code < 32u ? 1u << code : 0u;
        }
    }
    w.pv_init = low_mask<W>(m);
    w.x_init = w.pv_init + w.pv_init;
    w.m_mask = w.pv_init;
    w.rw = R.row_words;
    w.n = n;
    w.delta = delta;
    w.thr = p_valid ? P.l_max - delta : -1;
    w.l_max_lane = p_valid ? P.l_max : -1;
    w.l_max = P.l_max;
    w.lane = lane;
    w.p_sorted = R.p_start + p_rel;
    w.diag = R.diag;

    // codes of the bucket's level-1 nodes
    uint32_t root_codes = 0u;
    {
        const int cnt = (int)(R.root_end - R.root_begin);
        if (lane < cnt) root_codes = 1u << (P.trie[1][R.root_begin + lane].code & 31u);
        root_codes = __reduce_or_sync(kFull, root_codes);
    }
    visit<W, COUNT, 1>(w, P, R.root_begin, R.root_end, root_codes, w.pv_init, W(0));

    if (COUNT) {
        // warp-level counters (identical in all lanes): lane 0 reports 32 lanes' worth
        if (lane == 0) {
            atomicAdd(P.work + 0, w.n_cols * 32ull);
            atomicAdd(P.work + 1, w.n_tests * 32ull);
            atomicAdd(P.work + 2, w.n_first * 32ull);
            atomicAdd(P.work + 3, w.n_ptests * 32ull);
        }
    }
}

template <typename W, bool COUNT>
cudaError_t launch_one(const DistanceParams& p, int64_t n_items, size_t smem, cudaStream_t s) {
    auto kern = k_distance_trie<W, COUNT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<(unsigned)((n_items - p.shard + p.n_shards - 1) / p.n_shards), kTQ, smem, s>>>(p);
    return cudaGetLastError();
}

}  // namespace

size_t distance_trie_smem_bytes(bool wide) {
    const size_t peq = (size_t)kPeqRows * (wide ? peq_row_bytes<uint64_t>() : peq_row_bytes<uint32_t>());
    return peq + (size_t)(kTQ / 32) * kTrieDepth * kTrieFan * sizeof(uint4);
}

cudaError_t launch_distance_trie(const DistanceParams& p, int64_t n_items, bool wide, bool count_work,
                                 cudaStream_t s, int* launches) {
    if (n_items <= p.shard) return cudaSuccess;
    if (n_items > 0x7fffffffLL) return cudaErrorInvalidValue;
    const size_t smem = distance_trie_smem_bytes(wide);
    *launches += 1;
    if (wide)
        return count_work ? launch_one<uint64_t, true>(p, n_items, smem, s)
                          : launch_one<uint64_t, false>(p, n_items, smem, s);
    return count_work ? launch_one<uint32_t, true>(p, n_items, smem, s)
                      : launch_one<uint32_t, false>(p, n_items, smem, s);
}

}  // namespace tcrnet

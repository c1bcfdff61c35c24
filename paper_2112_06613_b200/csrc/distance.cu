// Steps A3-A5, text-chunk kernel: every length-compatible pair of one work item is visited.
//
// For every (pattern a of length m, text b of length n, m <= n <= m + l_max) of the item it decides
// lev(a,b) <= l_max exactly with the bit-parallel recurrence of myers.cuh.
//
// Mapping (B200: 4 SMSPs x 16-lane ALU pipe per SM): one CTA = 256 patterns (one per thread, its
// Peq column private in shared memory, layout Peq[code][thread] -> conflict-free) against a chunk
// of texts of ONE length, streamed through shared memory with 16-byte cp.async in a two-stage
// pipeline.  All 32 lanes of a warp work on the same text, so the column loop, the trip count and
// the early-exit branch are warp-uniform: no divergence.
//
// Early exit (step A4; "will abort, as soon as the smallest intermediate result
// exceeds" l_max): values never decrease along a DP diagonal and lev(a,b) is the last cell of the
// diagonal i - j = m - n, so after column j the cell D[j+m-n][j] is a lower bound of the distance
// (DESIGN.md section 4).  A warp leaves the column loop when that bound exceeds l_max in all 32
// lanes.  The result is identical with the test on or off.
//
// This kernel serves early-exit-off builds, prefix sharing off, and the buckets too short for the
// prefix-trie kernel (distance_trie.cu), which is the default for everything else.
#include "myers.cuh"

namespace tcrnet {
namespace {

// FIRST = text columns processed before the first early-exit test (0: early exit off).
// Hot path per (warp, text): one or two broadcast LDS.128 (the first 4 / 8 residue codes), FIRST
// unrolled columns, one test.  Everything else (remaining columns with a test every second column,
// the final distance, emission) is the cold path.
template <typename W, int FIRST, bool COUNT>
__global__ void __launch_bounds__(kTQ) k_distance(const __grid_constant__ DistanceParams P) {
    extern __shared__ __align__(16) unsigned char smem[];
    constexpr int kRowBytes = peq_row_bytes<W>();
    constexpr uint32_t kFull = 0xffffffffu;
    W* peq = reinterpret_cast<W*>(smem);
    uint32_t* tbuf = reinterpret_cast<uint32_t*>(smem + kPeqRows * kRowBytes);

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

    const int m = R.m, n = R.n, rw = R.row_words;
    const int delta = n - m;                  // 0 <= delta <= l_max
    const int l_max = P.l_max;

    const int p_rel = p_tile0 + tid;
    const bool p_valid = p_rel < R.p_count;
    build_peq<W>(peq, tid, p_valid, P.pat + (size_t)(R.p_start + p_rel) * P.pat_stride, m);

    const uint32_t smem_addr = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t lane_addr = smem_addr + tid * (uint32_t)sizeof(W);
    const uint32_t tbuf_addr = smem_addr + kPeqRows * kRowBytes;
    const W pv_init = low_mask<W>(m);
    W x_init = pv_init + pv_init;
    const W m_mask = pv_init;

    // the hot test: after FIRST columns, rows 1..FIRST-delta of the column (only if FIRST > delta, FIRST <= n)
    const bool hot = FIRST > 0 && FIRST <= n && FIRST > delta;
    const W first_mask = low_mask<W>(hot ? FIRST - delta : 0);
    int first_thr = l_max - FIRST;            // dead  <=>  popc(Pv & mask) - popc(Mv & mask) > first_thr
    // keep the loop invariants of the hot loop in registers (ptxas otherwise re-derives them per text)
    asm volatile("" : "+r"(first_thr));
    if (sizeof(W) == 4) {
        uint32_t x32 = (uint32_t)x_init;
        asm volatile("" : "+r"(x32));
        x_init = (W)x32;
    }

    // ---- text pipeline: kTT rows per stage, two stages, 16-byte cp.async ----
    const uint32_t* txt_chunk = P.txt + R.txt_base + (int64_t)chunk_t0 * rw;
    const int stage_words = kTT * rw;
    const int n_sub = (chunk_cnt + kTT - 1) / kTT;
    auto stage_load = [&](int sub) {
        const int cnt = min(kTT, chunk_cnt - sub * kTT);
        const uint4* src = reinterpret_cast<const uint4*>(txt_chunk + (int64_t)sub * stage_words);
        uint4* dst = reinterpret_cast<uint4*>(tbuf + (sub & 1) * stage_words);
        const int pieces = cnt * (rw >> 2);
        for (int k = tid; k < pieces; k += kTQ) cp_async16(dst + k, src + k);
    };

    unsigned long long n_cols = 0, n_tests = 0, n_first = 0;  // warp-level, COUNT only
    const int warp_p0 = p_tile0 + warp * 32;

    stage_load(0);
    cp_async_commit();
    for (int sub = 0; sub < n_sub; ++sub) {
        if (sub + 1 < n_sub) stage_load(sub + 1);
        cp_async_commit();
        cp_async_wait<1>();
        __syncthreads();

        const int sub_t0 = chunk_t0 + sub * kTT;
        const int cnt = min(kTT, chunk_cnt - sub * kTT);
        // same bucket: texts at or before this warp's first pattern pair with nobody (sorted p < t only)
        const int tt_begin = R.diag ? max(0, warp_p0 + 1 - sub_t0) : 0;
        const uint32_t row_bytes = (uint32_t)rw * 4u;
        uint32_t row_addr = tbuf_addr + (uint32_t)((sub & 1) * stage_words + tt_begin * rw) * 4u;
        // ---- cold path: the remaining columns (a test after every second one), distance, emission ----
        auto finish = [&](int tt, uint32_t row_addr, W Pv, W Mv, int j) {
            for (; j < n; ++j) {
                const W Eq = peq_load<W>(lane_addr, text_load1(row_addr + 4u * (uint32_t)j));
                column_step<W>(Eq, Pv, Mv);
                if (COUNT) ++n_cols;
                const int jj = j + 1;
                if (FIRST > 0 && (jj & 1) == 0 && jj > delta && jj < n) {
                    const W msk = low_mask<W>(jj - delta);
                    const int lb = jj + WordOps<W>::popc(Pv & msk) - WordOps<W>::popc(Mv & msk);
                    if (COUNT) ++n_tests;
                    if (!__any_sync(kFull, lb <= l_max)) return;
                }
            }
            const int d = n + WordOps<W>::popc(Pv & m_mask) - WordOps<W>::popc(Mv & m_mask);
            const int t_rel = sub_t0 + tt;
            const bool edge = d <= l_max && p_valid && (!R.diag || p_rel < t_rel);
            emit_edges(P, edge, lane, R.p_start + p_rel, R.t_start + t_rel, m, n);
        };
        if (hot) {
            // ---- hot loop: 1-2 broadcast LDS.128, FIRST unrolled columns, one warp-wide test ----
            for (int tt = tt_begin; tt < cnt; ++tt, row_addr += row_bytes) {
                uint32_t c[8];
                W Pv, Mv;
                text_load4(row_addr, c);
                if (FIRST > 4) text_load4(row_addr + 16u, c + 4);
                first_columns<W, FIRST>(lane_addr, c, pv_init, x_init, Pv, Mv);
                const int score = WordOps<W>::popc(Pv & first_mask) - WordOps<W>::popc(Mv & first_mask);
                if (COUNT) { ++n_first; n_cols += FIRST; ++n_tests; }
                if (__any_sync(kFull, score <= first_thr)) finish(tt, row_addr, Pv, Mv, FIRST);
            }
        } else {
            for (int tt = tt_begin; tt < cnt; ++tt, row_addr += row_bytes) finish(tt, row_addr, pv_init, W(0), 0);
        }
        __syncthreads();  // stage (sub & 1) is free for the load issued two iterations later
    }
    if (COUNT && lane == 0) {
        atomicAdd(P.work + 0, n_cols * 32ull);
        atomicAdd(P.work + 1, n_tests * 32ull);
        atomicAdd(P.work + 2, n_first * 32ull);
    }
}

template <typename W, int FIRST, bool COUNT>
cudaError_t launch_one(const DistanceParams& p, int64_t n_items, size_t smem, cudaStream_t s) {
    auto kern = k_distance<W, FIRST, COUNT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<(unsigned)((n_items - p.shard + p.n_shards - 1) / p.n_shards), kTQ, smem, s>>>(p);
    return cudaGetLastError();
}

template <typename W, bool COUNT>
cudaError_t launch_first(const DistanceParams& p, int64_t n_items, int first, size_t smem, cudaStream_t s) {
    switch (first) {
        case 0: return launch_one<W, 0, COUNT>(p, n_items, smem, s);
        case 3: return launch_one<W, 3, COUNT>(p, n_items, smem, s);
        case 4: return launch_one<W, 4, COUNT>(p, n_items, smem, s);
        case 5: return launch_one<W, 5, COUNT>(p, n_items, smem, s);
        case 6: return launch_one<W, 6, COUNT>(p, n_items, smem, s);
        case 7: return launch_one<W, 7, COUNT>(p, n_items, smem, s);
        case 8: return launch_one<W, 8, COUNT>(p, n_items, smem, s);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

size_t distance_smem_bytes(bool wide, int max_row_words) {
    const size_t peq = (size_t)kPeqRows * (wide ? peq_row_bytes<uint64_t>() : peq_row_bytes<uint32_t>());
    return peq + 2ull * kTT * max_row_words * sizeof(uint32_t);
}

cudaError_t launch_distance(const DistanceParams& p, int64_t n_items, bool wide, int first_check, bool count_work,
                            int max_row_words, cudaStream_t s, int* launches) {
    if (n_items <= p.shard) return cudaSuccess;
    if (n_items > 0x7fffffffLL) return cudaErrorInvalidValue;
    const size_t smem = distance_smem_bytes(wide, max_row_words);
    *launches += 1;
    if (wide)
        return count_work ? launch_first<uint64_t, true>(p, n_items, first_check, smem, s)
                          : launch_first<uint64_t, false>(p, n_items, first_check, smem, s);
    return count_work ? launch_first<uint32_t, true>(p, n_items, first_check, smem, s)
                      : launch_first<uint32_t, false>(p, n_items, first_check, smem, s);
}

}  // namespace tcrnet

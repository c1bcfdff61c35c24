// Steps A3-A5: the distance kernel.
//
// For every length-compatible pair (pattern a of length m, text b of length n, m <= n <= m+l_max)
// it decides lev(a,b) <= l_max exactly, with the bit-parallel column
// recurrence of Myers (1999) in Hyyro's (2001) formulation for the GLOBAL distance: the vertical
// deltas of one DP column live in two machine words, Pv (+1) and Mv (-1), bit i = row i+1.
//
//   D0  = (((Eq & Pv) + Pv) ^ Pv) | Eq | Mv          Eq = Peq[b_j], bit i set iff a_i == b_j
//   Hp  = Mv | ~(D0 | Pv)        Hn = Pv & D0
//   Pv' = (Hn << 1) | ~(D0 | ((Hp << 1) | 1))        the "| 1" is the boundary D[0][j] = j
//   Mv' = D0 & ((Hp << 1) | 1)
//
// and after column j:  D[i][j] = j + popc(Pv & low(i)) - popc(Mv & low(i))  for every row i,
// so lev(a,b) = n + popc(Pv & low(m)) - popc(Mv & low(m)) with no per-column score.
//
// We carry X = ~((Hp << 1) | 1) = (~Hp) << 1 instead of Hp: the boundary bit then costs
// nothing (X = nHp + nHp), and the negations fold into the LOP3 truth tables.  Per column and
// pair that is 7 LOP3 on the ALU pipe, 3 integer adds + 1 address IMAD that ptxas can place
// on the FMA pipe, and one 4-byte shared-memory load.
//
// Mapping (B200: 4 SMSPs x 16-lane ALU pipe per SM): one CTA = 256 patterns (one per thread,
// its Peq column private in shared memory, layout Peq[code][thread] -> conflict-free) against
// a chunk of texts of ONE length, streamed through shared memory with 16-byte cp.async in a
// two-stage pipeline.  All 32 lanes of a warp work on the same text, so the column loop, the
// trip count and the early-exit branch are warp-uniform: no divergence.
//
// Early exit (step A4; "will abort, as soon as the smallest intermediate result
// exceeds" l_max): values never decrease along a DP diagonal and lev(a,b) is the last cell of
// the diagonal i - j = m - n, so after column j the cell D[j+m-n][j] is a lower bound of the
// distance.  A warp leaves the column loop when that bound exceeds
// l_max in all 32 lanes.  The result is identical with the test on or off.
//
// Emission (step A5): __ballot_sync / __popc prefix, one atomicAdd per warp on the global
// cursor, keys (min(i,j) << 32) | max(i,j) in the caller's row numbering.
#include "tcrnet_internal.h"

namespace tcrnet {
namespace {

template <typename W>
struct WordOps;
template <>
struct WordOps<uint32_t> {
    static constexpr int kBits = 32;
    static constexpr int kRowPad = 4;  // words; row stride 1040 B is not a power of two (forces IMAD, not LEA)
    static __device__ __forceinline__ int popc(uint32_t x) { return __popc(x); }
};
template <>
struct WordOps<uint64_t> {
    static constexpr int kBits = 64;
    static constexpr int kRowPad = 2;
    static __device__ __forceinline__ int popc(uint64_t x) { return __popcll(x); }
};

template <typename W>
__device__ __forceinline__ W low_mask(int i) {  // i >= 0 low bits set
    return i >= WordOps<W>::kBits ? ~W(0) : ((W(1) << i) - W(1));
}

template <typename W>
__host__ __device__ constexpr int peq_row_bytes() {
    return (kTQ + WordOps<W>::kRowPad) * (int)sizeof(W);
}

template <typename W>
__device__ __forceinline__ void column_step(W Eq, W& Pv, W& Mv) {
    const W s = (Eq & Pv) + Pv;
    const W D0 = ((s ^ Pv) | Mv) | Eq;
    const W nHp = ~Mv & (D0 | Pv);  // ~Hp
    const W Hn = Pv & D0;
    const W X = nHp + nHp;          // ~((Hp << 1) | 1)
    const W Hn2 = Hn + Hn;          // Hn << 1
    Pv = Hn2 | (~D0 & X);
    Mv = D0 & ~X;
}

// K consecutive columns whose residue codes are c[0..K): all Peq loads first, then the chain.
template <typename W, int K>
__device__ __forceinline__ void columns(const unsigned char* lane_col, const uint32_t* c, W& Pv, W& Mv) {
    W Eq[K > 0 ? K : 1];
#pragma unroll
    for (int q = 0; q < K; ++q)
        Eq[q] = *reinterpret_cast<const W*>(lane_col + c[q] * (uint32_t)peq_row_bytes<W>());
#pragma unroll
    for (int q = 0; q < K; ++q) column_step<W>(Eq[q], Pv, Mv);
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}

template <typename W, int FIRST, bool COUNT>
__global__ void __launch_bounds__(kTQ) k_distance(const __grid_constant__ DistanceParams P) {
    extern __shared__ __align__(16) unsigned char smem[];
    constexpr int kRowBytes = peq_row_bytes<W>();
    constexpr uint32_t kFull = 0xffffffffu;
    W* peq = reinterpret_cast<W*>(smem);
    uint32_t* tbuf = reinterpret_cast<uint32_t*>(smem + kPeqRows * kRowBytes);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // ---- step A2, device side: which (bucket pair, pattern tile, text chunk) is this CTA? ----
    const int64_t item = blockIdx.x;
    int lo = 0, hi = P.n_rows;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (P.rows[mid].item_begin <= item) lo = mid; else hi = mid;
    }
    const WorkRow R = P.rows[lo];
    const int64_t local = item - R.item_begin;
    const int pi = (int)(local / R.n_tchunks), qi = (int)(local % R.n_tchunks);
    const int p_tile0 = pi * kTQ;             // relative to the pattern bucket
    const int chunk_t0 = qi * P.tchunk;       // relative to the text bucket
    const int chunk_cnt = min(P.tchunk, R.t_count - chunk_t0);
    if (R.diag && chunk_t0 + chunk_cnt <= p_tile0 + 1) return;  // wholly on/below the diagonal

    const int m = R.m, n = R.n, rw = R.row_words;
    const int delta = n - m;                  // 0 <= delta <= l_max
    const int l_max = P.l_max;

    // ---- Peq for this thread's pattern: column `tid` of peq[code][*] (private, no barrier) ----
    const int p_rel = p_tile0 + tid;
    const bool p_valid = p_rel < R.p_count;
#pragma unroll
    for (int r = 0; r < kPeqRows; ++r) peq[r * (kRowBytes / (int)sizeof(W)) + tid] = W(0);
    if (p_valid) {
        const uint4* prow = reinterpret_cast<const uint4*>(P.pat + (size_t)(R.p_start + p_rel) * P.pat_stride);
        for (int i0 = 0; i0 < m; i0 += 16) {
            const uint4 v = __ldg(prow + (i0 >> 4));
            const uint32_t w4[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                const int i = i0 + k;
                if (i < m) {
                    const uint32_t c = (w4[k >> 2] >> ((k & 3) * 8)) & 0xffu;
                    peq[c * (kRowBytes / (int)sizeof(W)) + tid] |= W(1) << i;
                }
            }
        }
    }
    const unsigned char* lane_col = smem + tid * (int)sizeof(W);
    const W pv_init = low_mask<W>(m);
    const W m_mask = pv_init;

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

    unsigned long long n_cols = 0, n_tests = 0, n_visits = 0;  // warp-level, COUNT only
    const int warp_p0 = p_tile0 + warp * 32;

    stage_load(0);
    cp_async_commit();
    for (int sub = 0; sub < n_sub; ++sub) {
        if (sub + 1 < n_sub) stage_load(sub + 1);
        cp_async_commit();
        cp_async_wait<1>();
        __syncthreads();

        const uint32_t* tb = tbuf + (sub & 1) * stage_words;
        const int cnt = min(kTT, chunk_cnt - sub * kTT);
        for (int tt = 0; tt < cnt; ++tt) {
            const int t_rel = chunk_t0 + sub * kTT + tt;
            if (R.diag && t_rel <= warp_p0) continue;  // every lane has p >= t
            const uint4* trow = reinterpret_cast<const uint4*>(tb + tt * rw);
            W Pv = pv_init, Mv = W(0);
            bool alive = true;
            int g = 0;
            if (COUNT) ++n_visits;

            // lower bound on the final diagonal after column j; only called with j > delta
            auto all_dead = [&](int j) -> bool {
                const W msk = low_mask<W>(j - delta);
                const int lb = j + WordOps<W>::popc(Pv & msk) - WordOps<W>::popc(Mv & msk);
                if (COUNT) ++n_tests;
                return !__any_sync(kFull, lb <= l_max);
            };

            if (FIRST > 0 && n >= 8) {
                const uint4 o0 = trow[0], o1 = trow[1];
                const uint32_t c[8] = {o0.x, o0.y, o0.z, o0.w, o1.x, o1.y, o1.z, o1.w};
                columns<W, FIRST>(lane_col, c, Pv, Mv);
                if (COUNT) n_cols += FIRST;
                if (FIRST > delta && all_dead(FIRST)) alive = false;
                if (alive) {
                    columns<W, 8 - FIRST>(lane_col, c + FIRST, Pv, Mv);
                    if (COUNT) n_cols += 8 - FIRST;
                    if (FIRST < 8 && 8 > delta && all_dead(8)) alive = false;
                }
                g = 2;
            }
            if (alive) {
                const int n_groups = n >> 2;
                for (; g < n_groups; ++g) {
                    const uint4 o = trow[g];
                    const uint32_t c[4] = {o.x, o.y, o.z, o.w};
                    columns<W, 4>(lane_col, c, Pv, Mv);
                    if (COUNT) n_cols += 4;
                    if (FIRST > 0) {
                        const int j = 4 * (g + 1);
                        if (j > delta && all_dead(j)) {
                            alive = false;
                            break;
                        }
                    }
                }
            }
            if (alive) {
                const int rem = n & 3;
                if (rem) {
                    const uint4 o = trow[n >> 2];
                    const uint32_t c[3] = {o.x, o.y, o.z};
                    if (rem == 1) columns<W, 1>(lane_col, c, Pv, Mv);
                    else if (rem == 2) columns<W, 2>(lane_col, c, Pv, Mv);
                    else columns<W, 3>(lane_col, c, Pv, Mv);
                    if (COUNT) n_cols += rem;
                }
                const int d = n + WordOps<W>::popc(Pv & m_mask) - WordOps<W>::popc(Mv & m_mask);
                const bool edge = d <= l_max && p_valid && (!R.diag || p_rel < t_rel);
                const uint32_t bal = __ballot_sync(kFull, edge);
                if (bal) {
                    unsigned long long base = 0;
                    if (lane == 0) base = atomicAdd(P.edge_count, (unsigned long long)__popc(bal));
                    base = __shfl_sync(kFull, base, 0);
                    if (edge) {
                        const unsigned long long pos = base + __popc(bal & ((1u << lane) - 1u));
                        if (pos < P.edge_cap) {
                            const uint32_t oi = (uint32_t)P.perm[R.p_start + p_rel];
                            const uint32_t oj = (uint32_t)P.perm[R.t_start + t_rel];
                            const uint32_t a = min(oi, oj), b = max(oi, oj);
                            P.edges[pos] = ((unsigned long long)a << 32) | b;
                        }
                    }
                }
            }
        }
        __syncthreads();  // stage (sub & 1) is free for the load issued two iterations later
    }
    if (COUNT && lane == 0) {
        atomicAdd(P.work + 0, n_cols * 32ull);
        atomicAdd(P.work + 1, n_tests * 32ull);
        atomicAdd(P.work + 2, n_visits * 32ull);
    }
}

template <typename W, int FIRST, bool COUNT>
cudaError_t launch_one(const DistanceParams& p, int64_t n_items, size_t smem, cudaStream_t s) {
    auto kern = k_distance<W, FIRST, COUNT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<(unsigned)n_items, kTQ, smem, s>>>(p);
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
    if (n_items <= 0) return cudaSuccess;
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

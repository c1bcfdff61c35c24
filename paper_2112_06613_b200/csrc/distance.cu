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

// lop3.b32 with an immediate truth table (a = 0xF0, b = 0xCC, c = 0xAA): written as PTX so that
// the front end cannot re-associate the recurrence into more LOP3s than the seven it needs.
template <int LUT>
__device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(r) : "r"(a), "r"(b), "r"(c), "n"(LUT));
    return r;
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

template <>
__device__ __forceinline__ void column_step<uint32_t>(uint32_t Eq, uint32_t& Pv, uint32_t& Mv) {
    const uint32_t t = lop3<0xC0>(Eq, Pv, 0u);        // Eq & Pv
    const uint32_t s = t + Pv;
    const uint32_t D0a = lop3<0xBE>(s, Pv, Mv);       // (s ^ Pv) | Mv
    const uint32_t D0 = lop3<0xFC>(D0a, Eq, 0u);      // | Eq
    const uint32_t nHp = lop3<0x0E>(Mv, D0, Pv);      // ~Mv & (D0 | Pv) = ~Hp
    const uint32_t Hn = lop3<0xC0>(Pv, D0, 0u);       // Pv & D0
    const uint32_t X = nHp + nHp;                     // ~((Hp << 1) | 1)
    const uint32_t Hn2 = Hn + Hn;                     // Hn << 1
    Pv = lop3<0xF2>(Hn2, D0, X);                      // Hn2 | (~D0 & X)
    Mv = lop3<0x30>(D0, X, 0u);                       // D0 & ~X
}

// Column 0 starts from Pv = low(m), Mv = 0.  Bits at and above m are don't-cares (they never flow
// down and are masked at every popcount), so ~Hp = D0 | Pv may be replaced by the constant Pv, and
// Hn = Pv & D0 by D0:  X = Pv0 + Pv0 is a constant and the step needs 3 LOP3 + 2 adds.
template <typename W>
__device__ __forceinline__ void first_column_step(W Eq, W Pv0, W X0, W& Pv, W& Mv) {
    const W s = Eq + Pv0;            // Eq & Pv0 = Eq: Peq has no bits at or above m
    const W D0 = ((s ^ Pv0) | Eq);
    const W Hn2 = D0 + D0;
    Pv = Hn2 | (~D0 & X0);
    Mv = D0 & ~X0;
}
template <>
__device__ __forceinline__ void first_column_step<uint32_t>(uint32_t Eq, uint32_t Pv0, uint32_t X0, uint32_t& Pv,
                                                             uint32_t& Mv) {
    const uint32_t s = Eq + Pv0;
    const uint32_t D0 = lop3<0xBE>(s, Pv0, Eq);       // (s ^ Pv0) | Eq
    const uint32_t Hn2 = D0 + D0;
    Pv = lop3<0xF2>(Hn2, D0, X0);                     // Hn2 | (~D0 & X0)
    Mv = lop3<0x30>(D0, X0, 0u);                      // D0 & ~X0
}

// Shared-memory accesses by 32-bit shared address (no generic-pointer arithmetic in the hot loop).
// The text loads are volatile so that they stay behind the barrier that publishes the stage; the Peq
// loads depend on their results.
template <typename W>
__device__ __forceinline__ W peq_load(uint32_t lane_addr, uint32_t code);
template <>
__device__ __forceinline__ uint32_t peq_load<uint32_t>(uint32_t lane_addr, uint32_t code) {
    uint32_t v;
    asm("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(lane_addr + code * (uint32_t)peq_row_bytes<uint32_t>()));
    return v;
}
template <>
__device__ __forceinline__ uint64_t peq_load<uint64_t>(uint32_t lane_addr, uint32_t code) {
    unsigned long long v;
    asm("ld.shared.u64 %0, [%1];" : "=l"(v) : "r"(lane_addr + code * (uint32_t)peq_row_bytes<uint64_t>()));
    return v;
}
__device__ __forceinline__ void text_load4(uint32_t addr, uint32_t* c) {
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(c[0]), "=r"(c[1]), "=r"(c[2]), "=r"(c[3]) : "r"(addr));
}
__device__ __forceinline__ uint32_t text_load1(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

// The first K columns of a text (codes c[0..K)): all Peq loads first, then the chain.
template <typename W, int K>
__device__ __forceinline__ void first_columns(uint32_t lane_addr, const uint32_t* c, W Pv0, W X0, W& Pv, W& Mv) {
    W Eq[K > 0 ? K : 1];
#pragma unroll
    for (int q = 0; q < K; ++q) Eq[q] = peq_load<W>(lane_addr, c[q]);
    if (K > 0) first_column_step<W>(Eq[0], Pv0, X0, Pv, Mv);
#pragma unroll
    for (int q = 1; q < K; ++q) column_step<W>(Eq[q], Pv, Mv);
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

// FIRST = text columns processed before the first early-exit test (0: early exit off).
// Hot path per (warp, text): one or two broadcast LDS.128 (the first 4 / 8 residue codes), FIRST unrolled
// columns, one test; ~95 % of the visits end there.  Everything else (remaining columns with a test every
// second column, the final distance, emission) is the cold path.
template <typename W, int FIRST, bool COUNT>
__global__ void __launch_bounds__(kTQ) k_distance(const __grid_constant__ DistanceParams P) {
    extern __shared__ __align__(16) unsigned char smem[];
    constexpr int kRowBytes = peq_row_bytes<W>();
    constexpr int kRowWords = kRowBytes / (int)sizeof(W);
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
    for (int r = 0; r < kPeqRows; ++r) peq[r * kRowWords + tid] = W(0);
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
                    peq[c * kRowWords + tid] |= W(1) << i;
                }
            }
        }
    }
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

    unsigned long long n_cols = 0, n_tests = 0, n_visits = 0;  // warp-level, COUNT only
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
                if (COUNT) { ++n_visits; n_cols += FIRST; ++n_tests; }
                if (__any_sync(kFull, score <= first_thr)) finish(tt, row_addr, Pv, Mv, FIRST);
            }
        } else {
            for (int tt = tt_begin; tt < cnt; ++tt, row_addr += row_bytes) {
                if (COUNT) ++n_visits;
                finish(tt, row_addr, pv_init, W(0), 0);
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

// Device helpers shared by the two distance kernels (distance.cu: text-chunk kernel,
// distance_trie.cu: prefix-trie kernel).  Internal to libtcrnet_b200.so; nothing here is shared with
// oracle/.
//
// The recurrence is the bit-parallel column step of Myers (1999) in Hyyro's (2001) formulation for
// the GLOBAL distance: the vertical deltas of one DP column live in two machine words, Pv (+1) and
// Mv (-1), bit i = row i+1.
//
//   D0  = (((Eq & Pv) + Pv) ^ Pv) | Eq | Mv          Eq = Peq[b_j], bit i set iff a_i == b_j
//   Hp  = Mv | ~(D0 | Pv)        Hn = Pv & D0
//   Pv' = (Hn << 1) | ~(D0 | ((Hp << 1) | 1))        the "| 1" is the boundary D[0][j] = j
//   Mv' = D0 & ((Hp << 1) | 1)
//
// and after column j:  D[i][j] = j + popc(Pv & low(i)) - popc(Mv & low(i))  for every row i,
// so lev(a,b) = n + popc(Pv & low(m)) - popc(Mv & low(m)) with no per-column score.
//
// We carry X = ~((Hp << 1) | 1) = (~Hp) << 1 instead of Hp: the boundary bit then costs nothing
// (X = nHp + nHp) and the negations fold into the LOP3 truth tables.  Per column and pair: 7 LOP3
// on the ALU pipe, 3 integer adds + 1 address IMAD that ptxas places on the FMA pipe, one 4-byte
// shared-memory load.
#pragma once

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

// Every step returns D0 (bit i set iff D[i+1][j] = D[i][j-1]: the diagonal did not increase), which the
// trie kernel uses to track the final-diagonal cell without popcounts.
template <typename W>
__device__ __forceinline__ W column_step(W Eq, W& Pv, W& Mv) {
    const W s = (Eq & Pv) + Pv;
    const W D0 = ((s ^ Pv) | Mv) | Eq;
    const W nHp = ~Mv & (D0 | Pv);  // ~Hp
    const W Hn = Pv & D0;
    const W X = nHp + nHp;          // ~((Hp << 1) | 1)
    const W Hn2 = Hn + Hn;          // Hn << 1
    Pv = Hn2 | (~D0 & X);
    Mv = D0 & ~X;
    return D0;
}

template <>
__device__ __forceinline__ uint32_t column_step<uint32_t>(uint32_t Eq, uint32_t& Pv, uint32_t& Mv) {
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
    return D0;
}

// Column 0 starts from Pv = low(m), Mv = 0.  Bits at and above m are don't-cares (they never flow
// down and are masked at every popcount), so ~Hp = D0 | Pv may be replaced by the constant Pv, and
// Hn = Pv & D0 by D0:  X = Pv0 + Pv0 is a constant and the step needs 3 LOP3 + 2 adds.
template <typename W>
__device__ __forceinline__ W first_column_step(W Eq, W Pv0, W X0, W& Pv, W& Mv) {
    const W s = Eq + Pv0;            // Eq & Pv0 = Eq: Peq has no bits at or above m
    const W D0 = ((s ^ Pv0) | Eq);
    const W Hn2 = D0 + D0;
    Pv = Hn2 | (~D0 & X0);
    Mv = D0 & ~X0;
    return D0;
}
template <>
__device__ __forceinline__ uint32_t first_column_step<uint32_t>(uint32_t Eq, uint32_t Pv0, uint32_t X0, uint32_t& Pv,
                                                                 uint32_t& Mv) {
    const uint32_t s = Eq + Pv0;
    const uint32_t D0 = lop3<0xBE>(s, Pv0, Eq);       // (s ^ Pv0) | Eq
    const uint32_t Hn2 = D0 + D0;
    Pv = lop3<0xF2>(Hn2, D0, X0);                     // Hn2 | (~D0 & X0)
    Mv = lop3<0x30>(D0, X0, 0u);                      // D0 & ~X0
    return D0;
}

// Shared-memory accesses by 32-bit shared address (no generic-pointer arithmetic in the hot loop).
// The text loads are volatile so that they stay behind the barrier that publishes the stage; the Peq
// loads depend on their results.
__device__ __forceinline__ void lds_word(uint32_t addr, uint32_t& v) { asm("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr)); }
__device__ __forceinline__ void lds_word(uint32_t addr, uint64_t& v) {
    unsigned long long t;
    asm("ld.shared.u64 %0, [%1];" : "=l"(t) : "r"(addr));
    v = t;
}
// Peq[code] of this thread's pattern; ROW_BYTES = bytes per Peq row (one word per pattern of the tile + padding)
template <typename W, int ROW_BYTES = peq_row_bytes<W>()>
__device__ __forceinline__ W peq_load(uint32_t lane_addr, uint32_t code) {
    W v;
    lds_word(lane_addr + code * (uint32_t)ROW_BYTES, v);
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

// Peq for this thread's pattern: column `tid` of peq[code][*] (private to the thread: no barrier).
template <typename W, int ROW_BYTES = peq_row_bytes<W>()>
__device__ __forceinline__ void build_peq(W* peq, int tid, bool p_valid, const uint8_t* pat_row, int m) {
    constexpr int kRowWords = ROW_BYTES / (int)sizeof(W);
#pragma unroll
    for (int r = 0; r < kPeqRows; ++r) peq[r * kRowWords + tid] = W(0);
    if (p_valid) {
        const uint4* prow = reinterpret_cast<const uint4*>(pat_row);
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
}

// Step A5: warp-aggregated emission of the pairs (pattern p_sorted, text t_sorted) with `edge` set.
// perm maps a sorted position to the caller's row.  When the load collapsed identical sequences (dedup.cu,
// P.group_start != NULL) it maps to the row of a sequence that only one row has, or to kGroupFlag | uid of a
// shared one; the pair is then only recorded here and k_expand_entries turns it into its (rows) x (rows) edges
// and does the counting.
__device__ __forceinline__ void emit_edges(const DistanceParams& P, bool edge, int lane, int p_sorted, int t_sorted,
                                           int m, int n) {
    uint32_t oi = 0, oj = 0;
    if (edge) {
        oi = (uint32_t)P.perm_p[p_sorted];
        oj = (uint32_t)P.perm_t[t_sorted];
        if (P.mode == kPairsQueryAll) edge = oj >= (uint32_t)P.n_query || n > m || oi < oj;
        else if (P.mode == kPairsAllQuery) edge = oi >= (uint32_t)P.n_query;
        else if (P.mode == kPairsSelfQuery) edge = min(oi, oj) < (uint32_t)P.n_query;
    }
    const uint32_t bal = __ballot_sync(0xffffffffu, edge);
    if (bal) {
        unsigned long long base = 0;
        if (lane == 0) base = atomicAdd(P.edge_count, (unsigned long long)__popc(bal));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (edge) {
            const unsigned long long pos = base + __popc(bal & ((1u << lane) - 1u));
            const uint32_t a = min(oi, oj), b = max(oi, oj);
            if (P.group_start == nullptr) {  // the keys are final: count them for the CSR step
                atomicAdd(P.row_count + a, 1);
                atomicAdd(P.deg + b, 1);
            }
            if (pos < P.edge_cap) P.edges[pos] = ((unsigned long long)a << 32) | b;
        }
    }
}

// Step A2, device side: the WorkRow that contains work item `item`.
__device__ __forceinline__ int64_t work_item(const DistanceParams& P) {  // step 8(e): interleaved shards
    return (int64_t)blockIdx.x * P.n_shards + P.shard;
}
__device__ __forceinline__ const WorkRow& find_row(const DistanceParams& P, int64_t item) {
    int lo = 0, hi = P.n_rows;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (P.rows[mid].item_begin <= item) lo = mid; else hi = mid;
    }
    return P.rows[lo];
}

}  // namespace
}  // namespace tcrnet

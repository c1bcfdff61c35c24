// Segment join: an exact candidate filter in front of steps A3-A5 (the tile scheduler of north_star (2) taken one
// step further: not only length-bucket pairs that cannot match are skipped, but every pair that shares no segment),
// and the banded verification of what it lets through.
//
// Pigeonhole: cut a text s (length n) into k = l_max + 1 consecutive segments.  An edit script of at most l_max
// operations touches at most l_max of them, so if lev(r, s) <= l_max at least one segment of s
// occurs UNCHANGED in r.  Take the first such segment, number i, starting at q in s and found at q + d in r
// (delta = n - |r| >= 0: the pattern r is the shorter sequence).  Each of the i segments before it holds at least
// one edit, the part before the match needs at least |d| insertions / deletions and the part after it at least
// |d + delta|, so   max(|d|, i) + |d + delta| <= l_max.   These (i, d) are the probes of JoinTables; everything else
// cannot be the first unchanged segment of a pair within l_max.  The filter has no false negatives.
//
// Layout: bit-plane rows (pack.cu).  Plane k of a sequence holds bit k of the 5-bit code of every residue, so for a
// diagonal s (text position = pattern position + s) the mismatch mask of a pair,
//      M_s[j] = (a_j != b_(j+s))  =  OR_k (A_k ^ (B_k >> s))[j],
// costs five shifts and five LOP3 for ALL residues at once.  Everything below works on these masks:
//
//   index   k_join_index: one entry (composition signature, text) per (text, segment), bucketed by a hash of
//           (n, i, segment bits) in a power-of-two directory (count -> prefix sum -> fill).
//   probe   k_join_probe: one warp = 32 patterns of one length x one length difference delta; for every probe each lane
//           hashes its pattern's substring; the 32 directory buckets are walked as ONE list, 32 entries per step; the
//           texts whose composition can be within l_max (same length bucket: only texts after the pattern in sorted
//           order, so every unordered pair is seen once) are queued in shared memory and checked 32 at a time, one per
//           lane: build the masks of the band's diagonals
//           s = -floor((l_max - delta) / 2) .. delta + floor((l_max - delta) / 2)  (no alignment with <= l_max edits
//           leaves the band) and apply
//             - the probe's own segment really matches (M restricted to it is zero: hash collisions die here),
//             - shifted-Hamming bound: a pattern residue that matches under NO diagonal of the band is substituted or
//               deleted in every alignment inside the band, so more than l_max of them means lev > l_max (exact as a
//               bound; kills nearly all random candidates),
//             - once: a pair can be found through several probes; it is kept by the FIRST probe (table order) whose
//               segment matches, which the masks decide without touching memory again.
//   verify  the survivors are decided exactly by Landau-Vishkin on the same masks: F[e][s] = the furthest pattern
//           position reachable on diagonal s with e edits; one step = max over (substitution, deletion, insertion)
//           followed by a slide over the zero run of M_s (count-trailing-zeros).  lev <= l_max iff F[l_max][delta]
//           reaches the end of the pattern.  This IS the banded early exit of step A4: cells outside the band are
//           never touched.  For l_max <= 1 it degenerates to the textbook check (equal lengths: at most one mismatch;
//           one longer: common prefix + common suffix cover the shorter sequence - SURVEY 8(f) NEXT-4) and runs
//           inline in the probe kernel; for l_max >= 2 the survivors are queued and k_join_verify applies the once
//           rule and then runs Landau-Vishkin densely, one lane per pair that is still there (the masks of a kept
//           pair wait with it in a shared-memory ring).
#include <algorithm>

#include "launch.cuh"
#include "myers.cuh"
#include "planes.cuh"

namespace tcrnet {
namespace {

constexpr uint32_t kFullMask = 0xffffffffu;
constexpr int kJoinWarps = 8;
constexpr int kJoinThreads = 32 * kJoinWarps;
constexpr int kProbeWarps = kJoinWarps;  // (CTAs of 4 warps, 12 per SM: no difference measured at configs 3-5)
constexpr int kProbeThreads = 32 * kProbeWarps;
constexpr int kUnreached = -1000;  // Landau-Vishkin: no alignment ends on this diagonal yet

// b seen from diagonal s: bit j of the result = bit j + s of b (zero outside)
template <typename W>
__device__ __forceinline__ W diag_shift(W b, int s) {
    return s >= 0 ? (b >> s) : (b << (-s));
}

template <typename W>
__device__ __forceinline__ int ctz_word(W x);
template <>
__device__ __forceinline__ int ctz_word<uint32_t>(uint32_t x) { return __ffs((int)x) - 1; }
template <>
__device__ __forceinline__ int ctz_word<uint64_t>(uint64_t x) { return __ffsll((long long)x) - 1; }

// from pattern position v on a diagonal with mask M: skip the run of matches (v <= lim <= bits of W; the bits of M
// at and beyond lim are set unless lim is the word size)
template <typename W>
__device__ __forceinline__ int slide(W M, int v, int lim) {
    if (v >= lim) return v;
    const W x = M >> v;
    const int adv = x ? ctz_word<W>(x) : WordOps<W>::kBits;
    return min(v + adv, lim);
}

// The band of a pair: diagonals smin .. smin + nb - 1 (nb <= L + 1).
__device__ __forceinline__ void band_of(int L, int delta, int& smin, int& nb) {
    const int h = (L - delta) >> 1;
    smin = -h;
    nb = delta + 2 * h + 1;
}

// bits of M_s that are set whatever the residues are: j >= m, or j + s outside the text
template <typename W>
__device__ __forceinline__ W invalid_mask(int s, int m, int n) {
    return ~(diag_shift<W>(low_mask<W>(n), s) & low_mask<W>(m));
}

// M_s: bit j set iff pattern residue j has NO equal partner on diagonal s (a_j != b_(j+s), or j >= m, or j + s
// outside the text).
// Mismatch masks of a band with the pair-independent parts given (probe kernel: the band is the same for all pairs of
// a warp): NV[x] = invalid_mask of diagonal x (all ones beyond the band).  32-bit planes: every plane of B is widened once
// (b << 8 as a 64-bit pair), after which any diagonal s in -8..23 is ONE funnel shift.
template <int L>
__device__ __forceinline__ void band_masks_hoisted(const PlaneRow<uint32_t>& A, const PlaneRow<uint32_t>& B, int smin,
                                                   const uint32_t (&NV)[L + 1], uint32_t (&M)[L + 1]) {
    uint32_t lo[5], hi[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) lo[k] = B.p[k] << 8, hi[k] = B.p[k] >> 24;
#pragma unroll
    for (int x = 0; x <= L; ++x) {
        uint32_t v = NV[x];
#pragma unroll
        for (int k = 0; k < 5; ++k) v |= A.p[k] ^ __funnelshift_r(lo[k], hi[k], (uint32_t)(8 + smin + x));
        M[x] = v;
    }
}
template <int L>
__device__ __forceinline__ void band_masks_hoisted(const PlaneRow<uint64_t>& A, const PlaneRow<uint64_t>& B, int smin,
                                                   const uint64_t (&NV)[L + 1], uint64_t (&M)[L + 1]) {
#pragma unroll
    for (int x = 0; x <= L; ++x) {
        uint64_t v = NV[x];
#pragma unroll
        for (int k = 0; k < 5; ++k) v |= A.p[k] ^ diag_shift<uint64_t>(B.p[k], smin + x);
        M[x] = v;
    }
}

// Mismatch masks of the band of ONE pair (verification kernel: every lane has its own m, n).
template <typename W, int L>
__device__ __forceinline__ void band_masks(const PlaneRow<W>& A, const PlaneRow<W>& B, int m, int n, int smin, int nb,
                                           W (&M)[L + 1]) {
    W NV[L + 1];
#pragma unroll
    for (int x = 0; x <= L; ++x) NV[x] = x < nb ? invalid_mask<W>(smin + x, m, n) : ~W(0);
    band_masks_hoisted<L>(A, B, smin, NV, M);
}

// shifted-Hamming bound: pattern residues without a partner on any diagonal of the band
template <typename W, int L>
__device__ __forceinline__ bool shd_pass(const W (&M)[L + 1], int m) {
    W u = M[0];
#pragma unroll
    for (int x = 1; x <= L; ++x) u &= M[x];
    return WordOps<W>::popc(u & low_mask<W>(m)) <= L;
}

template <typename W, int L>
__device__ __forceinline__ W mask_of_diag(const W (&M)[L + 1], int x) {  // M[x] without dynamic register indexing
    W r = ~W(0);
#pragma unroll
    for (int y = 0; y <= L; ++y)
        if (y == x) r = M[y];
    return r;
}

// the segment [sq, sq + len) of the text sits unchanged at [sq + d, sq + d + len) of the pattern (diagonal -d)
template <typename W, int L>
__device__ __forceinline__ bool segment_matches(const W (&M)[L + 1], int smin, int nb, int sq, int len, int d, int m) {
    const int rq = sq + d, x = -d - smin;
    if (rq < 0 || rq + len > m || x < 0 || x >= nb) return false;
    const W mk = mask_of_diag<W, L>(M, x);
    return ((mk >> rq) & low_mask<W>(len)) == W(0);
}

// Probe `pi` (text length n = m + delta) is the first of the table whose segment matches.
template <typename W, int L>
__device__ __forceinline__ bool first_matching_probe(const JoinTables& tab, const W (&M)[L + 1], int smin, int nb, int m,
                                                     int n, int delta, int pi) {
    for (int k = 0; k < pi; ++k) {
        const int i = tab.probe_seg[delta][k], d = tab.probe_shift[delta][k];
        const int sq = tab.seg_start[n][i], len = tab.seg_start[n][i + 1] - sq;
        if (segment_matches<W, L>(M, smin, nb, sq, len, d, m)) return false;
    }
    return true;
}

// Landau-Vishkin inside the band: true iff lev(a, b) <= L.
template <typename W, int L>
__device__ __forceinline__ bool lv_within(const W (&M)[L + 1], int m, int n, int delta, int smin, int nb) {
    int F[L + 1];
#pragma unroll
    for (int x = 0; x <= L; ++x) F[x] = (x == -smin) ? slide<W>(M[x], 0, m) : kUnreached;  // diagonal 0: lim = min(m, n) = m
#pragma unroll
    for (int e = 1; e <= L; ++e) {
        int G[L + 1];
#pragma unroll
        for (int x = 0; x <= L; ++x) {
            const int s = smin + x, lim = min(m, n - s);
            int v = F[x];
            if (v >= 0 && v < lim) v += 1;  // substitution of a_v by b_(v+s) (else: stay)
            if (x + 1 <= L) {               // deletion of a_u: from diagonal s + 1
                const int u = F[x + 1 <= L ? x + 1 : L];
                if (u >= 0 && u < m) v = max(v, u + 1);
            }
            if (x >= 1) {                   // insertion of b_(u+s-1): from diagonal s - 1
                const int u = F[x >= 1 ? x - 1 : 0];
                if (u >= 0 && u + s <= n) v = max(v, u);
            }
            G[x] = (x < nb && v >= 0) ? slide<W>(M[x], v, lim) : kUnreached;
        }
#pragma unroll
        for (int x = 0; x <= L; ++x) F[x] = G[x];
    }
    int end = kUnreached;
#pragma unroll
    for (int x = 0; x <= L; ++x)
        if (x == delta - smin) end = F[x];
    return end >= m;
}

// Composition signature of a sequence: the residue codes fall into 8 classes (code & 7); nibble g = the number of
// residues of class g, saturated at 7.  One edit moves at most one residue out of a class and one into a class, so
//     sum_g |count_r(g) - count_s(g)|  <=  2 * substitutions + insertions + deletions  <=  2 * l_max - delta
// for every pair within l_max whose lengths differ by delta (at least delta of the edits are insertions); saturation
// only shrinks the left side.  The index stores the signature of the text in every entry, so most texts that merely
// share a (short, low-entropy) segment with the pattern are dropped before their row is fetched.
template <typename W>
__device__ __forceinline__ uint32_t class_counts(const PlaneRow<W>& R) {
    const W valid = low_mask<W>(R.len);
    uint32_t sig = 0u;
#pragma unroll
    for (int g = 0; g < 8; ++g) {
        W mk = valid;
        mk &= (g & 1) ? R.p[0] : ~R.p[0];
        mk &= (g & 2) ? R.p[1] : ~R.p[1];
        mk &= (g & 4) ? R.p[2] : ~R.p[2];
        sig |= (uint32_t)min(WordOps<W>::popc(mk), 7) << (4 * g);
    }
    return sig;
}
// The top bit of every nibble is free: an index entry keeps its segment number there (bits 3, 7, 11), so that a probe
// for segment i only ever takes entries OF segment i.  Together with the residue-wise test of the probe's segment this
// makes a text appear at most once per probe: an entry of segment i that passes that test has the probe's key, and a
// text has one entry per segment (a foreign key that merely shares the hash bucket would otherwise let a text in twice).
__device__ __forceinline__ uint32_t segment_code(int i) {
    return (((uint32_t)i & 1u) << 3) | (((uint32_t)i & 2u) << 6) | (((uint32_t)i & 4u) << 9);
}
constexpr uint32_t kSegmentCodeMask = 0x888u;
// sum over the 8 nibbles of |a_g - b_g| (each 0..7; top bits of b ignored), SWAR
__device__ __forceinline__ int class_distance(uint32_t a, uint32_t b) {
    b &= 0x77777777u;
    const uint32_t x = (a | 0x88888888u) - b;                 // nibble g = 8 + a_g - b_g: no borrow leaves a nibble
    const uint32_t neg = (~x >> 3) & 0x11111111u;             // 1 where a_g < b_g
    uint32_t v = (x ^ (neg * 7u)) & 0x77777777u;              // |a_g - b_g| - [a_g < b_g]
    v = (v & 0x0F0F0F0Fu) + ((v >> 4) & 0x0F0F0F0Fu);
    return (int)((v * 0x01010101u) >> 24) + __popc(neg);
}

// hash of (text length n, segment i, residues [q, q + len) of the row): 32-bit arithmetic throughout (the directory has
// at most 2^30 slots; a collision only lets a foreign key into a bucket, where the residue-wise tests drop it)
__device__ __forceinline__ uint32_t fold32(uint32_t x) { return x; }
__device__ __forceinline__ uint32_t fold32(uint64_t x) { return (uint32_t)x ^ ((uint32_t)(x >> 32) * 0x9E3779B1u); }
template <typename W>
__device__ __forceinline__ uint32_t seg_hash(const PlaneRow<W>& R, int q, int len, int n, int i) {
    uint32_t h = (uint32_t)(n * 8 + i) * 0x9E3779B1u + 0x7F4A7C15u;
    const W mk = low_mask<W>(len);
#pragma unroll
    for (int k = 0; k < 5; ++k) h = (h ^ fold32((R.p[k] >> q) & mk)) * 0x85EBCA6Bu + 0xC2B2AE35u;
    h ^= h >> 16;  // (murmur3's finaliser: the low bits select the slot)
    h *= 0x85EBCA6Bu;
    h ^= h >> 13;
    h *= 0xC2B2AE35u;
    h ^= h >> 16;
    return h;
}

// ---- index ----
template <typename W, bool FILL>
__global__ void __launch_bounds__(256) k_join_index(const void* __restrict__ planes, int64_t n,
                                                   const __grid_constant__ JoinTables tab, uint32_t* __restrict__ cnt,
                                                   const uint32_t* __restrict__ dir, uint2* __restrict__ entries,
                                                   uint32_t mask) {
    grid_dependency_wait();
    const int k = tab.n_seg;
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t t = idx / k;
    const int i = (int)(idx - t * k);
    if (t >= n) return;
    const PlaneRow<W> R = load_planes<W>(planes, t);
    if (R.len < k) return;  // too short to be cut into k segments: such buckets stay with the other kernels
    const int q = tab.seg_start[R.len][i], len = tab.seg_start[R.len][i + 1] - q;
    const uint32_t b = seg_hash<W>(R, q, len, R.len, i) & mask;
    if (!FILL) {
        atomicAdd(cnt + b, 1u);
    } else {
        const uint32_t slot = atomicSub(cnt + b, 1u) - 1u;
        entries[dir[b] + slot] = make_uint2(class_counts<W>(R) | segment_code(i), (uint32_t)t);
    }
}

// ---- probe ----
struct JoinParams {
    DistanceParams d;  // emission, n_items, shard
    JoinRowDev rows[kJoinMaxRows];  // (in the parameter block: no upload, no global loads in the row search)
    int32_t n_rows;
    int32_t pad_;
    int64_t n_local;                // work items of this shard
    const void* planes;
    JoinIndex index;
    uint2* cand;                    // l_max >= 2: (pattern, text) pairs that passed the filters ...
    uint8_t* cand_probe;            // ... and the probe that found each
    unsigned long long* cand_count; // keeps counting beyond cand_cap
    unsigned long long cand_cap;
    JoinTables tab;
};

__device__ __forceinline__ const JoinRowDev& find_join_row(const JoinParams& S, int64_t item) {
    int lo = 0, hi = S.n_rows;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if ((int64_t)S.rows[mid].item_begin <= item) lo = mid; else hi = mid;
    }
    return S.rows[lo];
}

// Per-warp staging in shared memory: the texts found by the bucket walks wait in `queue` until 32 of them can be
// checked at once, one per lane (the walks themselves keep few lanes busy: buckets differ in length and most lanes
// find nothing in a given step); what passes waits in `out` until 32 results leave with ONE atomic on the global
// cursor (edge list for l_max <= 1, verification queue beyond).
static_assert(kJoinMaxProbes <= 64, "queue entries keep the probe in 6 bits");
constexpr int kWin = 2;              // windows of 32 list positions per step of the bucket walk (join kernels at
                                     // config 5: 4.17 ms with 1, 3.83 with 2, 4.18 with 4 - registers)
constexpr int kQueue = 64 * kWin;    // ring: < 32 waiting + kWin windows (a power of two)
template <typename W>
struct WarpBuf {
    W a[5][32];          // [plane][lane]: the 32 patterns of the warp (registers are scarcer than shared memory here)
    W nv[8];             // invalid_mask of every diagonal of the band (the same for all pairs of the warp)
    uint4 bucket[32];    // the non-empty buckets of the current probe: (first entry, entries, signature, pattern lane)
                         // on the low slots; .x becomes first entry - start in the walked list
    uint2 queue[kQueue]; // ring: (owner lane | probe << 5 | segment code of the entry << 12, text)
    uint2 out[64];       // (pattern, text), sorted positions
    uint8_t out_probe[64];
};

template <typename W, int L, bool COUNT>
struct ProbeWarp {
    WarpBuf<W>* wb;
    int lane, p0;   // sorted position of lane 0's pattern
    int m, n, delta, smin, nb;
    int qhead = 0, qn = 0, on = 0;
    unsigned long long n_pass = 0, n_diag = 0;
};

// the first 32 staged results leave
template <typename W, int L, bool COUNT>
__device__ __forceinline__ void flush_out(ProbeWarp<W, L, COUNT>& w, const JoinParams& S, int cnt) {
    const bool act = w.lane < cnt;
    const uint2 pt = act ? w.wb->out[w.lane] : make_uint2(0u, 0u);
    const uint32_t pr = act ? w.wb->out_probe[w.lane] : 0u;
    uint2 rest = make_uint2(0u, 0u);
    uint32_t rest_pr = 0u;
    const bool mv = cnt + w.lane < w.on;  // what stays moves to the front
    if (mv) rest = w.wb->out[cnt + w.lane], rest_pr = w.wb->out_probe[cnt + w.lane];
    __syncwarp();
    if (mv) w.wb->out[w.lane] = rest, w.wb->out_probe[w.lane] = (uint8_t)rest_pr;
    w.on -= cnt;
    __syncwarp();
    if (L <= 1) {
        emit_edges(S.d, act, w.lane, (int)pt.x, (int)pt.y, w.m, w.n);
    } else {
        unsigned long long base = 0;
        if (w.lane == 0) base = atomicAdd(S.cand_count, (unsigned long long)cnt);
        base = __shfl_sync(kFullMask, base, 0);
        if (act && base + w.lane < S.cand_cap) {
            S.cand[base + w.lane] = pt;
            S.cand_probe[base + w.lane] = (uint8_t)pr;
        }
    }
}

// the first cnt queued texts are checked, one per lane
template <typename W, int L, bool COUNT>
__device__ __forceinline__ void drain_round(ProbeWarp<W, L, COUNT>& w, const JoinParams& S, int cnt) {
    const bool act = w.lane < cnt;
    const uint2 q = act ? w.wb->queue[(w.qhead + w.lane) & (kQueue - 1)] : make_uint2(0u, 0u);
    w.qhead = (w.qhead + cnt) & (kQueue - 1);
    w.qn -= cnt;
    if (COUNT) w.n_diag += (unsigned long long)(cnt * w.nb);  // mismatch masks built (warp-level count)
    const int ow = (int)(q.x & 31u), pi = (int)((q.x >> 5) & 63u), t = (int)q.y;
    PlaneRow<W> Ao;  // the owner's pattern
    W NV[L + 1];
#pragma unroll
    for (int k = 0; k < 5; ++k) Ao.p[k] = w.wb->a[k][ow];
#pragma unroll
    for (int x = 0; x <= L; ++x) NV[x] = w.wb->nv[x];
    bool keep = false;
    if (act) {
        const PlaneRow<W> B = load_planes<W>(S.planes, t);
        // (an entry of another length bucket that shares the hash bucket could not pass the segment test below either)
        if (B.len == w.n) {
            W M[L + 1];
            band_masks_hoisted<L>(Ao, B, w.smin, NV, M);
            const int i = S.tab.probe_seg[w.delta][pi], d = S.tab.probe_shift[w.delta][pi];
            const int sq = S.tab.seg_start[w.n][i], len = S.tab.seg_start[w.n][i + 1] - sq;
            // (the entry belongs to the probe's segment - a foreign key that shares the hash bucket does not)
            keep = ((q.x >> 12) & kSegmentCodeMask) == segment_code(i) && shd_pass<W, L>(M, w.m) &&
                   segment_matches<W, L>(M, w.smin, w.nb, sq, len, d, w.m);
            if (COUNT && keep) ++w.n_pass;
            if (L <= 1 && keep)
                keep = first_matching_probe<W, L>(S.tab, M, w.smin, w.nb, w.m, w.n, w.delta, pi) &&
                       lv_within<W, L>(M, w.m, w.n, w.delta, w.smin, w.nb);
        }
    }
    const uint32_t bal = __ballot_sync(kFullMask, keep);
    if (keep) {
        const int pos = w.on + __popc(bal & ((1u << w.lane) - 1u));
        w.wb->out[pos] = make_uint2((uint32_t)(w.p0 + ow), (uint32_t)t);
        w.wb->out_probe[pos] = (uint8_t)pi;
    }
    w.on += __popc(bal);
    __syncwarp();
    if (w.on >= 32) flush_out<W, L, COUNT>(w, S, 32);
}

// One warp = 32 consecutive patterns of one length x the texts longer by delta: every probe of that delta in turn.
// (Register cap for 5 / 6 CTAs per SM: the kernel waits on dependent L2 reads, warps hide more than a few spills cost -
// measured at config 5: 7.35 -> 7.08 ms per step.)
template <typename W, int L, bool COUNT>
__global__ void __launch_bounds__(kProbeThreads, (L >= 5 ? 4 : L >= 2 ? 6 : 5))
k_join_probe(const __grid_constant__ JoinParams S) {
    grid_dependency_wait();
    __shared__ WarpBuf<W> bufs[kProbeWarps];
    const DistanceParams& P = S.d;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t local = (int64_t)blockIdx.x * kProbeWarps + warp;
    if (local >= S.n_local) return;  // the whole warp
    const int64_t item = local * P.n_shards + P.shard;
    const JoinRowDev& Rw = find_join_row(S, item);
    const int rel = (int)(item - (int64_t)Rw.item_begin);
    const int tile = rel / (L + 1), delta = rel - tile * (L + 1);
    if (!((Rw.t_mask >> delta) & 1u)) return;  // no texts of that length
    ProbeWarp<W, L, COUNT> w;
    w.wb = &bufs[warp];
    w.lane = lane;
    w.m = Rw.m;
    w.n = w.m + delta;
    w.delta = delta;
    band_of(L, delta, w.smin, w.nb);
#pragma unroll
    for (int x = 0; x <= L; ++x)
        if (lane == x) w.wb->nv[x] = x < w.nb ? invalid_mask<W>(w.smin + x, w.m, w.n) : ~W(0);
    w.p0 = Rw.p_start + tile * 32;
    const bool p_valid = tile * 32 + lane < Rw.p_count;
    const int p = p_valid ? w.p0 + lane : w.p0;
    uint32_t sig;
    {
        const PlaneRow<W> A = load_planes<W>(S.planes, p);
        sig = class_counts<W>(A);
#pragma unroll
        for (int k = 0; k < 5; ++k) w.wb->a[k][lane] = A.p[k];
    }
    __syncwarp();
    const int sig_max = 2 * L - delta;  // composition bound of a pair within L
    const int m = w.m, n = w.n;
    unsigned long long n_entries = 0, n_cand = 0, n_probes = 0;
    uint32_t lt_mask, le_mask;  // (special registers: one instruction wherever the compiler re-creates them)
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(lt_mask));
    asm("mov.u32 %0, %%lanemask_le;" : "=r"(le_mask));

    const int np = S.tab.n_probes[delta];
    for (int pi = 0; pi < np; ++pi) {
        const int i = S.tab.probe_seg[delta][pi], d = S.tab.probe_shift[delta][pi];
        const int sq = S.tab.seg_start[n][i], len = S.tab.seg_start[n][i + 1] - sq, rq = sq + d;
        if (rq < 0 || rq + len > m) continue;  // the segment does not fit at this shift (warp-uniform)
        uint32_t e = 0, e_end = 0;
        if (p_valid) {
            PlaneRow<W> A;
#pragma unroll
            for (int k = 0; k < 5; ++k) A.p[k] = w.wb->a[k][lane];
            const uint32_t b = seg_hash<W>(A, rq, len, n, i) & S.index.mask;
            e = __ldg(S.index.dir + b);
            e_end = __ldg(S.index.dir + b + 1);
        }
        if (COUNT) n_probes += (unsigned long long)__popc(__ballot_sync(kFullMask, p_valid));
        // The 32 buckets are walked as ONE list, 32 entries per step whatever their lengths.  The non-empty buckets are
        // moved to the low lanes (their starts in the list are then strictly increasing); in every step the buckets that
        // start inside the current window of 32 positions mark their start in one mask (one warp-wide OR), and a
        // position's bucket is the number of starts at or before it.
        const int c = (int)(e_end - e);
        const uint32_t nz = __ballot_sync(kFullMask, c > 0);
        if (!nz) continue;
        if (c > 0) w.wb->bucket[__popc(nz & lt_mask)] = make_uint4(e, (uint32_t)c, sig, (uint32_t)lane);
        __syncwarp();
        const int c_k = lane < __popc(nz) ? (int)w.wb->bucket[lane].y : 0;  // entries of bucket `lane`
        int incl = c_k;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(kFullMask, incl, o);
            if (lane >= o) incl += v;
        }
        const int total = __shfl_sync(kFullMask, incl, 31);
        const int first = c_k ? incl - c_k : 0x7fffffff;  // position of this bucket's first entry in the list
        if (c_k) w.wb->bucket[lane].x -= (uint32_t)first;  // list position f of this bucket = entry .x + f
        __syncwarp();
        if (COUNT) n_entries += (unsigned long long)total;
        int before = 0;  // buckets that start before the window
        // kWin windows per step: all their entry reads are in flight before the first is looked at
        for (int f0 = 0; f0 < total; f0 += 32 * kWin) {
            uint2 cur[kWin];
            uint32_t sig_o[kWin];
            int ow[kWin];  // the lane whose pattern probes the bucket
            bool in[kWin];
#pragma unroll
            for (int u = 0; u < kWin; ++u) {
                const int f = f0 + 32 * u + lane;
                const uint32_t rel = (uint32_t)(first - (f0 + 32 * u));
                const uint32_t starts = __reduce_or_sync(kFullMask, rel < 32u ? 1u << rel : 0u);
                const int src = before + __popc(starts & le_mask) - 1;  // (position 0 starts bucket 0: never negative)
                before += __popc(starts);
                const uint4 bo = w.wb->bucket[src];
                sig_o[u] = bo.z;
                ow[u] = (int)bo.w;
                in[u] = f < total;
                cur[u] = make_uint2(0u, 0u);
                if (in[u]) cur[u] = __ldg(S.index.entries + (uint32_t)(bo.x + (uint32_t)f));  // (32-bit wrap intended)
            }
#pragma unroll
            for (int u = 0; u < kWin; ++u) {
                // composition bound; same length bucket: only the texts after the pattern (every unordered pair once).
                // (An entry of ANOTHER segment that merely shares the hash bucket is dropped by drain_round.)
                const bool has = in[u] && class_distance(sig_o[u], cur[u].x) <= sig_max &&
                                 (delta > 0 || (int)cur[u].y > w.p0 + ow[u]);
                const uint32_t bal = __ballot_sync(kFullMask, has);
                if (has) w.wb->queue[(w.qhead + w.qn + __popc(bal & lt_mask)) & (kQueue - 1)] = make_uint2(
                             (uint32_t)ow[u] | ((uint32_t)pi << 5) | ((cur[u].x & kSegmentCodeMask) << 12), cur[u].y);
                const int cq = __popc(bal);
                w.qn += cq;
                if (COUNT) n_cand += (unsigned long long)cq;
            }
            __syncwarp();
            while (w.qn >= 32) drain_round<W, L, COUNT>(w, S, 32);
        }
    }
    if (w.qn > 0) drain_round<W, L, COUNT>(w, S, w.qn);
    if (w.on > 0) flush_out<W, L, COUNT>(w, S, w.on);
    if (COUNT) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) w.n_pass += __shfl_xor_sync(kFullMask, w.n_pass, o);
        if (lane == 0) {
            atomicAdd(P.work + 5, n_probes);
            atomicAdd(P.work + 6, n_entries);
            atomicAdd(P.work + 7, n_cand);
            atomicAdd(P.work + 4, w.n_pass);
            atomicAdd(P.work + 0, w.n_diag);
        }
    }
}

// ---- verify (l_max >= 2): one lane per surviving pair ----
// Two steps, each at full lane occupancy: (1) every lane takes a queued pair, builds the mismatch masks of its band and
// applies the *once* rule (most of the queue are pairs found through several probes: only the first matching probe
// keeps its find); what is kept waits - masks included - in a per-warp ring in shared memory until (2) 32 pairs can run
// Landau-Vishkin together.
template <typename W, int L>
struct VerifyRing {
    uint2 pt[64];       // (pattern, text), sorted positions
    W M[L + 1][64];     // mismatch masks of the band
    uint16_t mn[64];    // m | n << 8
};

template <typename W, int L, bool COUNT>
__global__ void __launch_bounds__(kJoinThreads) k_join_verify(const __grid_constant__ JoinParams S) {
    grid_dependency_wait();
    __shared__ VerifyRing<W, L> rings[kJoinWarps];
    const DistanceParams& P = S.d;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    VerifyRing<W, L>& q = rings[warp];
    int qhead = 0, qn = 0;
    const unsigned long long total = min(*S.cand_count, S.cand_cap);
    unsigned long long n_edges = 0, n_diag = 0;
    auto lv_round = [&](int cnt) {  // the first cnt kept pairs, one per lane
        const bool act = lane < cnt;
        const int slot = (qhead + lane) & 63;
        qhead = (qhead + cnt) & 63;
        qn -= cnt;
        uint2 pt = make_uint2(0u, 0u);
        int m = 0, n = 0;
        bool edge = false;
        if (act) {
            pt = q.pt[slot];
            m = q.mn[slot] & 0xff, n = q.mn[slot] >> 8;
            W M[L + 1];
#pragma unroll
            for (int x = 0; x <= L; ++x) M[x] = q.M[x][slot];
            int smin, nb;
            band_of(L, n - m, smin, nb);
            edge = lv_within<W, L>(M, m, n, n - m, smin, nb);
        }
        if (COUNT && edge) ++n_edges;
        emit_edges(P, edge, lane, (int)pt.x, (int)pt.y, m, n);
        __syncwarp();  // (the slots are free again)
    };
    for (unsigned long long base = (unsigned long long)blockIdx.x * kJoinThreads; base < total;
         base += (unsigned long long)gridDim.x * kJoinThreads) {
        const unsigned long long c = base + threadIdx.x;
        bool keep = false;
        uint2 pt = make_uint2(0u, 0u);
        W M[L + 1];
        int m = 0, n = 0;
        if (c < total) {
            pt = S.cand[c];
            const int pi = (int)S.cand_probe[c];
            const PlaneRow<W> A = load_planes<W>(S.planes, pt.x);
            const PlaneRow<W> B = load_planes<W>(S.planes, pt.y);
            m = A.len, n = B.len;
            int smin, nb;
            band_of(L, n - m, smin, nb);
            band_masks<W, L>(A, B, m, n, smin, nb, M);
            if (COUNT) n_diag += (unsigned long long)nb;
            // once: only the first probe whose segment matches keeps the pair
            keep = first_matching_probe<W, L>(S.tab, M, smin, nb, m, n, n - m, pi);
        }
        const uint32_t bal = __ballot_sync(kFullMask, keep);
        if (keep) {
            const int slot = (qhead + qn + __popc(bal & ((1u << lane) - 1u))) & 63;
            q.pt[slot] = pt;
            q.mn[slot] = (uint16_t)(m | (n << 8));
#pragma unroll
            for (int x = 0; x <= L; ++x) q.M[x][slot] = M[x];
        }
        qn += __popc(bal);
        __syncwarp();
        if (qn >= 32) lv_round(32);
    }
    if (qn > 0) lv_round(qn);
    if (COUNT) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            n_edges += __shfl_xor_sync(kFullMask, n_edges, o);
            n_diag += __shfl_xor_sync(kFullMask, n_diag, o);
        }
        if (lane == 0 && n_diag) {
            atomicAdd(P.work + 3, n_edges);
            atomicAdd(P.work + 0, n_diag);
        }
    }
}

template <typename W, int L>
cudaError_t launch_join_l(const JoinParams& S, bool count_work, int n_sm, cudaStream_t s, int* launches) {
    const unsigned blocks = (unsigned)((S.n_local + kProbeWarps - 1) / kProbeWarps);
    if (count_work) launch_dep(k_join_probe<W, L, true>, blocks, kProbeThreads, 0, s, S);
    else launch_dep(k_join_probe<W, L, false>, blocks, kProbeThreads, 0, s, S);
    *launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess || L <= 1) return e;
    const unsigned vblocks = (unsigned)(n_sm * 8);
    if (count_work) launch_dep(k_join_verify<W, (L >= 2 ? L : 2), true>, vblocks, kJoinThreads, 0, s, S);
    else launch_dep(k_join_verify<W, (L >= 2 ? L : 2), false>, vblocks, kJoinThreads, 0, s, S);
    *launches += 1;
    return cudaGetLastError();
}

template <typename W>
cudaError_t launch_join_w(const JoinParams& S, bool count_work, int n_sm, cudaStream_t s, int* launches) {
    switch (S.d.l_max) {
        case 0: return launch_join_l<W, 0>(S, count_work, n_sm, s, launches);
        case 1: return launch_join_l<W, 1>(S, count_work, n_sm, s, launches);
        case 2: return launch_join_l<W, 2>(S, count_work, n_sm, s, launches);
        case 3: return launch_join_l<W, 3>(S, count_work, n_sm, s, launches);
        case 4: return launch_join_l<W, 4>(S, count_work, n_sm, s, launches);
        case 5: return launch_join_l<W, 5>(S, count_work, n_sm, s, launches);
        case 6: return launch_join_l<W, 6>(S, count_work, n_sm, s, launches);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

cudaError_t launch_join_index(const void* planes, bool wide, const LengthTable& lt, int64_t n, const JoinTables& tab,
                              uint32_t* cnt, uint32_t* dir, uint2* entries, uint32_t slots, void* scan_scratch,
                              cudaStream_t s, int* launches) {
    (void)lt;
    const int64_t threads = n * tab.n_seg;
    if (threads <= 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((threads + 255) / 256);
    if (wide) launch_dep(k_join_index<uint64_t, false>, blocks, 256, 0, s, planes, n, tab, cnt, nullptr, nullptr,
                         slots - 1u);
    else launch_dep(k_join_index<uint32_t, false>, blocks, 256, 0, s, planes, n, tab, cnt, nullptr, nullptr,
                    slots - 1u);
    *launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    e = exclusive_scan_u32_total(cnt, dir, (int64_t)slots, scan_scratch, s, launches);
    if (e != cudaSuccess) return e;
    if (wide) launch_dep(k_join_index<uint64_t, true>, blocks, 256, 0, s, planes, n, tab, cnt, dir, entries,
                         slots - 1u);
    else launch_dep(k_join_index<uint32_t, true>, blocks, 256, 0, s, planes, n, tab, cnt, dir, entries, slots - 1u);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_join(const DistanceParams& p, const JoinRow* rows, int n_rows, const void* planes, bool wide,
                        const JoinIndex& index, const JoinTables& tab, uint2* cand, uint8_t* cand_probe,
                        unsigned long long* cand_count, unsigned long long cand_cap, bool count_work, int n_sm,
                        cudaStream_t s, int* launches) {
    if (p.n_items <= p.shard || n_rows <= 0) return cudaSuccess;
    JoinParams S{};
    S.d = p;
    if (n_rows > kJoinMaxRows || p.n_items > 0xffffffffLL) return cudaErrorInvalidValue;
    for (int r = 0; r < n_rows; ++r) {  // rows: host memory
        JoinRowDev& d = S.rows[r];
        d.item_begin = (uint32_t)rows[r].item_begin;
        d.p_start = rows[r].p_start;
        d.p_count = rows[r].p_count;
        d.m = (uint8_t)rows[r].m;
        d.t_mask = 0;
        for (int q = 0; q < kJoinMaxSeg; ++q)
            if (rows[r].t_count[q] > 0) d.t_mask |= (uint8_t)(1u << q);
    }
    S.n_rows = n_rows;
    S.planes = planes;
    S.index = index;
    S.cand = cand;
    S.cand_probe = cand_probe;
    S.n_local = (p.n_items - p.shard + p.n_shards - 1) / p.n_shards;
    S.cand_count = cand_count;
    S.cand_cap = cand_cap;
    S.tab = tab;
    return wide ? launch_join_w<uint64_t>(S, count_work, n_sm, s, launches)
                : launch_join_w<uint32_t>(S, count_work, n_sm, s, launches);
}

}  // namespace tcrnet

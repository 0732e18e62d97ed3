// S8..S12: GESR serving selection (Eq. 13-14 + fallback), per-token
// communication cost (App. C), per-partition load, the decayed load state
// (Eq. 15, once per micro-batch per north_star / Q19) and fairness
// (Eq. 17-18).
//
// The evaluation is split where the data dependence is:
//
//   eval_scan_kernel   everything that does NOT depend on the load snapshot, at streaming speed and
//                      without any wait: persistent CTAs walk items = (layer, micro-batch, slice of
//                      <= 32768 tokens); per token the primary map is looked up in a 16-bit table, the
//                      slots of experts without replicas are counted (lane-private shared-memory
//                      counters, no branch) and, when the token has no replicated slot, its communication
//                      cost is final.  A token WITH replicated slots leaves one 16-byte record (accessed
//                      set so far | the rank of the replicated expert in each slot | home, family,
//                      offset).  Every item writes one row of partial sums
//                      (loads | span | remote | tokens per family | records).
//   eval_chain_kernel  the serial part (replicas only): one thread-block cluster per layer walks the
//                      micro-batches in order: snapshot -> guard -> sorted candidate tables of the
//                      replicated experts -> the records of the micro-batch (each pending slot takes the
//                      first local candidate of its table, else the first) -> integer dispatch counts,
//                      exchanged over distributed shared memory with one cluster barrier per
//                      micro-batch -> Eq. 15 applied redundantly by every CTA from the same integers
//                      (same fp64 operations, same bits; no floating-point value crosses a CTA).
//   fairness_kernel    S12; without replicas it first adds the rows of a layer (nothing depends on
//                      the snapshot then, the whole trace is one micro-batch).
//
// The only waits between CTAs are cluster barriers (a cluster is co-scheduled by the hardware) and, when one
// layer gets more CTAs than a cluster holds (few layers, long micro-batches: kModeGrid), a per-layer arrival
// counter inside a COOPERATIVE launch, where every CTA is resident by construction.
//
// tacg_eval_primary_noalloc (end of the file) runs the no-replica evaluation with the item rows in a fixed
// __device__ array instead of the context's scratch: an entry point that allocates nothing.
//
// The pick rule of Q17 orders candidates by (not local, snapshot load, candidate slot).  Only the
// first key depends on the token, so once per micro-batch each replicated expert's feasible
// candidates are sorted by (snapshot load, slot) into a small table; a token then takes the first
// entry that is local to it (in its accessed set R or its home), else the first entry.  That is
// the same argmin, with all fp64 comparisons hoisted out of the token loop.
//
// Shapes outside the record format (k not in {2,4,6,8} or an unaligned trace, more than 15 replicated
// experts in a layer) mark their items "overflow": the chain kernel then serves those tokens itself,
// straight from the trace.
#include <cooperative_groups.h>

#include <algorithm>
#include <type_traits>
#include <map>
#include <mutex>
#include <tuple>

#include "tacg_common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int kEvalThreads = 512;    // eval_scan_kernel, select_kernel
constexpr int kEvalBatch = 4;        // tokens per thread with their loads in flight together
constexpr int kSlice = 32768;        // most tokens of a scan item (64 per thread).  Bounded by the packed sums: a thread's
                                     // 11-bit span field (74 tokens x 16), the 16-bit record counts of an item, the chain
                                     // kernel's 16-bit per-thread fields over a round of 32 slices
constexpr int kOffBits = 15;         // record meta word: offset in the item (kOffBits) | family (3) | home partition (6)
static_assert(kSlice <= (1 << kOffBits), "record offsets");
constexpr int kChainThreads = 512;    // two CTAs per SM, so that clusters of 4 at L = 58 still use every SM
constexpr unsigned kRecFlight = 4;    // records a chain thread loads before it resolves the first (cluster, single CTA)
constexpr unsigned kRecFlightGrid = 1; // the same in grid mode, where a thread has one or two records per micro-batch
constexpr long long kSeqBelow = 1024; // micro-batches shorter than this go to the one-warp-per-layer kernel
constexpr int kCandStride = 12;      // bytes per expert in the candidate table: [0] = count, [1..9] = partitions
constexpr unsigned kRepFlag = 0x80u; // ptab bit: the expert has at least one replica
constexpr unsigned kBadFlag = 0x40u; // ptab bit: not an expert (empty slot, id outside [0,E))
constexpr int kPtab = 516;           // ids are clamped to 512; entry 512 is "not an expert"
constexpr int kSink = 64;            // counter row of the slots the scan kernel does not count
constexpr int kMaxRank = 15;         // replicated experts per layer the 4-bit rank fields can name
constexpr unsigned kCntAlign = 16384u;  // eval_scan_kernel's counter block (see there)
constexpr unsigned kT16Bad = 0x10u;     // tab16 entry: row << 7 (bits 7..13) | rank (bits 0..3) | kT16Bad
constexpr unsigned kOverflow = 0xffffffffu;   // record count of an item the chain kernel serves from the trace

struct LayerTables {
    unsigned char* ptab;   // [kPtab] primary partition | kRepFlag, or kBadFlag
    unsigned char* cand;   // [E][kCandStride] sorted feasible candidates of replicated experts
    signed char* rep;      // [E*r] replica partitions as given, -1 = none
    double* S;             // [64] load snapshot
};

__device__ __forceinline__ void load_ptab(int E, int r, const int8_t* __restrict__ pr, const int8_t* __restrict__ rp,
                                          unsigned char* ptab, signed char* rep) {
    for (int e = threadIdx.x; e < kPtab; e += blockDim.x) {
        unsigned v = kBadFlag;
        if (e < E) {
            unsigned n = 0;
            for (int a = 0; a < r; ++a) {
                const signed char c = rp[(size_t)e * r + a];
                if (rep) rep[e * r + a] = c;
                n += (c >= 0) ? 1u : 0u;
            }
            v = ((unsigned)pr[e] & 63u) | (n ? kRepFlag : 0u);
        }
        ptab[e] = (unsigned char)v;
    }
}

// Ranks of the replicated experts of a layer: 1, 2, ... in increasing expert id (0 = not replicated).
// Needs ptab complete (a barrier before); `wsum` is scratch for blockDim/32 words; ends with a barrier.
// Returns the number of replicated experts.  rank8[e] is clipped to 255; replist[rank-1] = e (optional).
__device__ __forceinline__ int build_ranks(int E, const unsigned char* ptab, unsigned char* rank8,
                                           unsigned short* replist, unsigned* wsum) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nw = blockDim.x >> 5;
    int base = 0;
    for (int e0 = 0; e0 < E; e0 += blockDim.x) {
        const int e = e0 + tid;
        const bool isrep = e < E && (ptab[e] & kRepFlag);
        const unsigned b = __ballot_sync(0xffffffffu, isrep);
        if (lane == 0) wsum[warp] = __popc(b);
        __syncthreads();
        int before = base;
        for (int q = 0; q < warp; ++q) before += (int)wsum[q];
        int total = 0;
        for (int q = 0; q < nw; ++q) total += (int)wsum[q];
        if (e < E) {
            const int rk = isrep ? before + __popc(b & ((1u << lane) - 1u)) + 1 : 0;
            rank8[e] = (unsigned char)min(rk, 255);
            if (isrep && replist) replist[rk - 1] = (unsigned short)e;
        }
        base += total;
        __syncthreads();
    }
    return base;
}

// feas from a snapshot: mean summed left to right in double (Q19), theta widened from float.
__device__ __forceinline__ unsigned long long load_guard(const double* S, int P, float theta) {
    double tot = 0.0;
    for (int m = 0; m < P; ++m) tot = __dadd_rn(tot, S[m]);
    const double Lbar = tot / (double)P;
    const double thr = __dmul_rn(__dadd_rn(1.0, (double)theta), Lbar);
    unsigned long long fm = 0ull;
    for (int m = 0; m < P; ++m)
        if (S[m] <= thr) fm |= 1ull << m;
    return fm;
}

// Candidate table entry of one replicated expert for one snapshot: the candidates (primary, then
// replicas in slot order), restricted to the feasible ones unless none is (fallback,
// PAPER.md:155), stably sorted by snapshot load (strict <, so ties keep slot order).
// out: [0] = count, [1..count] = partitions, entries up to [3] repeat [1] (pick_first3 reads three).
__device__ __forceinline__ void build_candidate(int e, int r, const LayerTables& T, unsigned long long feas,
                                                unsigned char* out) {
    const unsigned in = T.ptab[e];
    int c[9];
    int n = 0;
    c[n++] = (int)(in & 63u);
    for (int a = 0; a < r; ++a) {
        const int v = T.rep[e * r + a];
        if (v >= 0) c[n++] = v & 63;
    }
    unsigned long long cmask = 0ull;
    for (int i = 0; i < n; ++i) cmask |= 1ull << c[i];
    const bool anyfeas = (cmask & feas) != 0ull;
    int m = 0;
    for (int i = 0; i < n; ++i) {
        if (anyfeas && !((feas >> c[i]) & 1ull)) continue;
        // insertion: after every entry whose load is <= this one's
        const double s = T.S[c[i]];
        int pos = m;
        while (pos > 0 && s < T.S[out[pos]]) { out[pos + 1] = out[pos]; --pos; }
        out[pos + 1] = (unsigned char)c[i];
        ++m;
    }
    out[0] = (unsigned char)m;
    for (int i = m + 1; i <= 3; ++i) out[i] = out[1];
}

// load_guard by one whole warp: the same left-to-right fp64 sum (every lane computes it, eight independent loads at a
// time in front of the dependent additions), then one ballot per 32 partitions instead of a loop.  S has 64 entries.
__device__ __forceinline__ unsigned long long load_guard_warp(const double* S, int P, float theta, int lane) {
    double tot = 0.0;
    for (int m0 = 0; m0 < P; m0 += 8) {
        double v[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = S[min(m0 + i, 63)];
#pragma unroll
        for (int i = 0; i < 8; ++i)
            if (m0 + i < P) tot = __dadd_rn(tot, v[i]);
    }
    // P a power of two: tot * 2^-k is the same real number as tot / 2^k, so the rounded result is the same bits, without
    // the division's long dependent sequence
    const double Lbar = (P & (P - 1)) == 0 ? __dmul_rn(tot, 1.0 / (double)P) : tot / (double)P;
    const double thr = __dmul_rn(__dadd_rn(1.0, (double)theta), Lbar);
    unsigned long long fm = __ballot_sync(0xffffffffu, lane < P && S[lane] <= thr);
    if (P > 32) fm |= (unsigned long long)__ballot_sync(0xffffffffu, lane + 32 < P && S[lane + 32] <= thr) << 32;
    return fm;
}

// build_candidate for r <= 3 (at most four candidates) without a data-dependent loop: the position of a candidate in
// the stable order is the number of kept candidates that are lighter, or as heavy and earlier in slot order.
// The loads are compared through order_key: integer compares instead of fp64 ones, the same order.
__device__ __forceinline__ unsigned long long order_key(double x) {
    // -0.0 + 0.0 = +0.0, so equal loads have equal keys; then the usual map of IEEE bits onto unsigned order
    const long long b = __double_as_longlong(__dadd_rn(x, 0.0));
    return (unsigned long long)b ^ ((unsigned long long)(b >> 63) | 0x8000000000000000ull);
}

// The table entry is returned in two words: w0 = count | c1 << 8 | c2 << 16 | c3 << 24 (entries beyond the count repeat
// c1), w1 = c4.
__device__ __forceinline__ void build_candidate_small(int e, int r, const LayerTables& T, const unsigned long long* K,
                                                      unsigned long long feas, unsigned& w0, unsigned& w1) {
    int c[4];
    bool ok[4];
    c[0] = (int)(T.ptab[e] & 63u);
    ok[0] = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int v = a < r ? (int)T.rep[e * r + a] : -1;
        ok[a + 1] = v >= 0;
        c[a + 1] = v & 63;
    }
    unsigned long long cmask = 0ull;
#pragma unroll
    for (int i = 0; i < 4; ++i)
        if (ok[i]) cmask |= 1ull << c[i];
    const bool anyfeas = (cmask & feas) != 0ull;
    unsigned long long s[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        ok[i] = ok[i] && (!anyfeas || ((feas >> c[i]) & 1ull));
        s[i] = K[c[i]];
    }
    unsigned b[4] = {0u, 0u, 0u, 0u};      // partitions by position
    int m = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        int pos = 0;
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (j != i && ok[j] && (s[j] < s[i] || (j < i && s[j] == s[i]))) ++pos;
        if (ok[i]) {
            ++m;
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (pos == q) b[q] = (unsigned)c[i];
        }
    }
    if (m < 2) b[1] = b[0];
    if (m < 3) b[2] = b[0];
    if (m < 4) b[3] = b[0];
    w0 = (unsigned)m | (b[0] << 8) | (b[1] << 16) | (b[2] << 24);
    w1 = b[3];
}

// The same in three steps for the chain kernel, where one lane owns one replicated expert for a whole layer:
//   cand_fixed   once per layer: the candidates (one byte each, primary first), which of them exist, their partition set
//   cand_order   per micro-batch, BEFORE the guard is known (it only needs the loads): bit 4*i + j = candidate j sorts
//                before candidate i (lighter, or as heavy and earlier in slot order)
//   cand_tables  per micro-batch, after the guard: drop the infeasible ones (unless none is feasible), positions by
//                counting, table words as build_candidate_small returns them
struct CandFixed {
    unsigned cpk, okm;
    unsigned long long cmask;
};
__device__ __forceinline__ CandFixed cand_fixed(int e, int r, const LayerTables& T) {
    CandFixed f;
    f.cpk = T.ptab[e] & 63u;
    f.okm = 1u;
    f.cmask = 1ull << (T.ptab[e] & 63u);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int v = a < r ? (int)T.rep[e * r + a] : -1;
        if (v >= 0) {
            f.cpk |= (unsigned)(v & 63) << (8 * (a + 1));
            f.okm |= 1u << (a + 1);
            f.cmask |= 1ull << (v & 63);
        }
    }
    return f;
}
__device__ __forceinline__ unsigned cand_order(unsigned cpk, const unsigned long long* K) {
    unsigned long long s[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) s[i] = K[(cpk >> (8 * i)) & 63u];
    unsigned bef = 0u;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (j != i && (s[j] < s[i] || (j < i && s[j] == s[i]))) bef |= 1u << (4 * i + j);
    return bef;
}
__device__ __forceinline__ void cand_tables(const CandFixed& f, unsigned bef, unsigned long long feas, unsigned& w0,
                                            unsigned& w1) {
    unsigned okf = f.okm;
    if (f.cmask & feas) {
#pragma unroll
        for (int i = 0; i < 4; ++i)
            if (!((feas >> ((f.cpk >> (8 * i)) & 63u)) & 1ull)) okf &= ~(1u << i);
    }
    const int m = __popc(okf);
    unsigned bb = 0u;                       // partitions by position, one byte each
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int pos = __popc(okf & (bef >> (4 * i)) & 15u);
        if ((okf >> i) & 1u) bb |= ((f.cpk >> (8 * i)) & 0xffu) << (8 * pos);
    }
    // positions beyond the count repeat the first
    const unsigned keep = m >= 4 ? 0xffffffffu : (1u << (8 * m)) - 1u;
    bb = (bb & keep) | (((bb & 0xffu) * 0x01010101u) & ~keep);
    w0 = (unsigned)m | (bb << 8);
    w1 = bb >> 24;
}

__device__ __forceinline__ void build_candidates(int E, int r, const LayerTables& T, unsigned long long feas) {
    for (int e = threadIdx.x; e < E; e += blockDim.x)
        if (T.ptab[e] & kRepFlag) build_candidate(e, r, T, feas, T.cand + e * kCandStride);
}

// One pending (replicated) slot: the first candidate of the expert's sorted table that is local to the
// token (in R or its home), else the first.
template <typename M>
__device__ __forceinline__ int pick_candidate(const unsigned char* __restrict__ c, M loc) {
    const int n = c[0];
    int pick = c[1];
    for (int i = 1; i <= n; ++i) {
        const int v = c[i];
        if ((loc >> v) & (M)1) { pick = v; break; }
    }
    return pick;
}

// The same pick on the table's first word (count | c1 | c2 | c3, entries beyond the count repeat c1): no loop
// unless more than three candidates are listed and none of the first three is local.
template <typename M>
__device__ __forceinline__ int pick_first3(const unsigned char* __restrict__ c, M loc) {
    const unsigned w0 = *reinterpret_cast<const unsigned*>(c);
    const unsigned c1 = (w0 >> 8) & 0xffu, c2 = (w0 >> 16) & 0xffu, c3 = w0 >> 24;
    const bool l1 = (loc >> c1) & (M)1, l2 = (loc >> c2) & (M)1, l3 = (loc >> c3) & (M)1;
    int pick = l1 ? (int)c1 : (l2 ? (int)c2 : (l3 ? (int)c3 : (int)c1));
    if (!(l1 | l2 | l3) && (w0 & 0xffu) > 3u) {
        const int n = (int)(w0 & 0xffu);
        for (int i = 4; i <= n; ++i) {
            const int v = c[i];
            if ((loc >> v) & (M)1) { pick = v; break; }
        }
    }
    return pick;
}

// Step 4 of O10 for one token: serve[j] per slot (-1 = empty), returns the accessed set R.
template <int KM, typename M = unsigned long long>
__device__ __forceinline__ M serve_token(const int (&e)[KM], int k, int E, int home, const LayerTables& T,
                                         int (&sv)[KM]) {
    M R = 0;
    unsigned pending = 0u;
    // pass 1: experts with a single candidate are served by their primary regardless (Q18)
#pragma unroll
    for (int j = 0; j < KM; ++j) {
        sv[j] = -1;
        if (j < k && (unsigned)e[j] < (unsigned)E) {
            const unsigned in = T.ptab[e[j]];
            if (!(in & kRepFlag)) {
                sv[j] = (int)in;
                R |= (M)1 << in;
            } else {
                pending |= 1u << j;
            }
        }
    }
    // pass 2: replicated experts in slot order
    const M hb = (M)1 << home;
#pragma unroll
    for (int j = 0; j < KM; ++j) {
        if (!((pending >> j) & 1u)) continue;
        const int pick = pick_candidate<M>(T.cand + e[j] * kCandStride, R | hb);
        sv[j] = pick;
        R |= (M)1 << pick;
    }
    return R;
}

// ---- geometry shared by the scan and the chain kernels
struct EvalGeom {
    long long N, B, nmb, token_offset;
    long long ipl;      // items per layer = nmb * spm
    int spm;            // slices per micro-batch
    int slice;          // tokens per slice: a multiple of 512, <= kSlice
    int W;              // 32-bit words per row: P loads | F span | F remote | F tokens per family | records with one
                        // pending slot | records with several
    int k, L, E, F, P, r;
};

__device__ __forceinline__ void item_tokens(const EvalGeom& g, long long mb, int s, long long& t0, long long& t1) {
    t0 = mb * g.B + (long long)s * g.slice;
    const long long e = min(g.N, (mb + 1) * g.B);
    t1 = min(e, t0 + g.slice);
    if (t1 < t0) t1 = t0;
}

// Records of the deferred tokens of an item, g.slice 16-byte entries per item (tokens with one pending slot from entry
// 0 upwards, tokens with several from the last entry downwards), one load or store each:
//   x, y  accessed set after pass 1 (partitions of the slots without replicas), low and high word
//   z     4 bits per slot: rank of the replicated expert in that slot, 0 = not pending
//   w     offset in the item (13) | family (3) | home (6)
typedef uint4 Rec;
template <typename M> __device__ __forceinline__ Rec make_rec(M R, unsigned rank, unsigned meta) {
    return make_uint4((unsigned)R, (unsigned)((unsigned long long)R >> 32), rank, meta);
}
template <typename M> __device__ __forceinline__ M rec_set(const Rec& v) {
    if constexpr (sizeof(M) == 8) return (unsigned long long)v.x | ((unsigned long long)v.y << 32);
    else return v.x;
}

// 1 << s with PTX semantics: a shift count >= the register width gives 0 (the sink row 64 is no partition)
template <typename M> __device__ __forceinline__ M bit_or_zero(unsigned s);
template <> __device__ __forceinline__ unsigned bit_or_zero<unsigned>(unsigned s) {
    unsigned r;
    asm("shl.b32 %0, 1, %1;" : "=r"(r) : "r"(s));
    return r;
}
template <> __device__ __forceinline__ unsigned long long bit_or_zero<unsigned long long>(unsigned s) {
    unsigned long long r;
    asm("shl.b64 %0, 1, %1;" : "=l"(r) : "r"(s));
    return r;
}

// shared-memory accesses by 32-bit shared-space address (no generic-address arithmetic in the token loop)
__device__ __forceinline__ unsigned saddr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
// The same address, opaque to the compiler: it stays in its register instead of being recomputed (special-register reads
// and address arithmetic) at every use inside the hot loops.
__device__ __forceinline__ unsigned saddr_kept(const void* p) {
    unsigned a = saddr(p);
    asm volatile("" : "+r"(a));
    return a;
}
__device__ __forceinline__ void sred_inc(unsigned a) { asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(a) : "memory"); }
__device__ __forceinline__ void sred_add(unsigned a, unsigned v) {
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned slds_u32(unsigned a) {
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ unsigned slds_u8(unsigned a) {
    unsigned v;
    asm("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ unsigned slds_u16(unsigned a) {
    unsigned short v;
    asm("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a));
    return (unsigned)v;
}

struct ScanParams {
    EvalGeom g;
    const int16_t* indices;
    const int8_t* family;
    const int8_t* primary;
    const int8_t* replicas;   // null: no replicas
    unsigned* rows;           // [L*ipl][W]
    Rec* rec;                 // [L*ipl][slice] (replicas only)
    unsigned char* cost;      // [L,N] or null
    signed char* serve;       // [L,N,k] or null
};

template <typename M> __device__ __forceinline__ int popc_m(M x);
template <> __device__ __forceinline__ int popc_m<unsigned>(unsigned x) { return __popc(x); }
template <> __device__ __forceinline__ int popc_m<unsigned long long>(unsigned long long x) { return __popcll(x); }

// KT: compile-time k (0 = generic), REP: a replica table is present, M: partition-set mask type
// (unsigned for P <= 32, else unsigned long long), OUT: per-token outputs were requested.
template <int KT, bool REP, typename M, bool OUT>
__global__ void __launch_bounds__(kEvalThreads, 2) eval_scan_kernel(const ScanParams p) {
    tacg_pdl_prologue();
    constexpr int KM = KT > 0 ? KT : 16;
    constexpr int NW = KT > 0 ? KT / 2 : 1;
    constexpr int U = KT > 0 ? kEvalBatch : 1;
    constexpr bool RECS = REP && KT > 0;      // the record format covers compile-time k only
    extern __shared__ __align__(16) unsigned char esm[];
    // [65][32] lane-private columns, row 64 = sink; on a 16 KB boundary of the shared window, so that a counter's address
    // is (table entry & 0x3f80) | column address: one LOP3 per slot
    unsigned* cnt = reinterpret_cast<unsigned*>(esm + ((kCntAlign - (saddr(esm) & (kCntAlign - 1u))) & (kCntAlign - 1u)));
    unsigned* accb = cnt + (kSink + 1) * 32;                               // [warps][8][32] per-thread family words
    __shared__ unsigned char ptab[kPtab];
    __shared__ unsigned char rank8[kPtab];
    __shared__ unsigned short tab16[kPtab];   // row << 7 | rank | kT16Bad: the row field is the counter row's byte offset
    __shared__ unsigned comm_s[16];           // span[8] | remote[8] of this item
    __shared__ unsigned fam_s[8];
    __shared__ unsigned wsum[kEvalThreads / 32 + 1];
    __shared__ unsigned nrec_s;

    const EvalGeom& g = p.g;
    const int tid = threadIdx.x, lane = tid & 31;
    const int P = g.P, k = KT > 0 ? KT : g.k, E = g.E, F = g.F;
    const long long T = (long long)g.L * g.ipl;
    const long long lo = (long long)blockIdx.x * T / gridDim.x, hi = (long long)(blockIdx.x + 1) * T / gridDim.x;
    const unsigned cl = saddr_kept(cnt + lane);                             // this lane's counter column
    unsigned* acc = accb + (tid >> 5) * (8 * 32) + lane;                    // this thread's family words
    const unsigned al = saddr_kept(acc);
    const unsigned tb = saddr(tab16), pb8 = saddr(ptab), nrb = saddr(&nrec_s);
    // A thread's tokens of an item are S apart, S the largest multiple of P not above the CTA size (448..512): the home
    // partition (token index mod P) of all of them is the same, no per-token update.  The kEvalThreads % P last threads
    // idle when P does not divide the CTA size (no configuration of the paper).
    const int S = kEvalThreads - kEvalThreads % P;
    const bool worker = tid < S;

    for (int i = tid; i < (kSink + 1) * 32; i += kEvalThreads) cnt[i] = 0u;
#pragma unroll
    for (int f = 0; f < 8; ++f) acc[f * 32] = 0u;
    int cur_layer = -1;
    bool layer_ovf = REP && !RECS;           // this layer's items are left to the chain kernel
    // (layer, micro-batch, slice) of the first item by division, of the following ones by counting
    int layer = (int)(lo / g.ipl);
    long long mb = (lo - (long long)layer * g.ipl) / g.spm;
    int sl = (int)(lo - (long long)layer * g.ipl - mb * g.spm);
    int hm0 = (int)((g.token_offset + mb * g.B + (long long)sl * g.slice) % P);   // home of the item's first token
    const int hstep = g.slice % P;
    for (long long item = lo; item < hi; ++item) {
        __syncthreads();                    // the previous item's row is written
        if (layer != cur_layer) {
            load_ptab(E, REP ? g.r : 0, p.primary + (size_t)layer * E,
                      REP ? p.replicas + (size_t)layer * E * g.r : nullptr, ptab, nullptr);
            __syncthreads();
            int nrep = 0;
            if constexpr (REP) nrep = build_ranks(E, ptab, rank8, nullptr, wsum);
            layer_ovf = REP && (!RECS || nrep > kMaxRank);
            for (int e = tid; e < kPtab; e += kEvalThreads) {
                const unsigned v = ptab[e];
                unsigned t16;
                if (v & kBadFlag) t16 = (kSink << 7) | kT16Bad;
                else if (v & kRepFlag) t16 = (kSink << 7) | (REP ? (unsigned)rank8[e] & 15u : 0u);
                else t16 = (v & 63u) << 7;
                tab16[e] = (unsigned short)t16;
            }
            cur_layer = layer;
        }
        if (tid < 16) comm_s[tid] = 0u;
        if (tid < 8) fam_s[tid] = 0u;
        if (tid == 0) nrec_s = 0u;
        __syncthreads();
        long long t0, t1;
        item_tokens(g, mb, sl, t0, t1);
        const int n = (int)(t1 - t0);
        const int16_t* base = p.indices + (size_t)layer * (size_t)g.N * (size_t)k;
        unsigned char* cost_l = (OUT && p.cost) ? p.cost + (size_t)layer * g.N + t0 : nullptr;
        signed char* serve_l = (OUT && p.serve) ? p.serve + ((size_t)layer * g.N + t0) * k : nullptr;
        Rec* recs = RECS ? p.rec + (size_t)item * g.slice : nullptr;
        asm volatile("" : "+l"(recs));      // kept in its register pair: otherwise rebuilt from item and slice per record
        const int home = (hm0 + tid) % P;
        const int8_t* fam0 = p.family + t0;
        const unsigned* rows0 = reinterpret_cast<const unsigned*>(base + (size_t)t0 * k);   // KT > 0 only

        for (int ob = tid; ob < n + tid; ob += S * U) {      // uniform trip count across the CTA
            int f[U];
            unsigned w[U][NW];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int o = ob + u * S;
                f[u] = -1;
                if (worker && o < n) {
                    f[u] = fam0[o];
                    if constexpr (KT == 8) {
                        const uint4 v = __ldg(reinterpret_cast<const uint4*>(rows0) + o);
                        w[u][0] = v.x; w[u][1] = v.y; w[u][2] = v.z; w[u][3] = v.w;
                    } else if constexpr (KT == 4) {
                        const uint2 v = __ldg(reinterpret_cast<const uint2*>(rows0) + o);
                        w[u][0] = v.x; w[u][1] = v.y;
                    } else if constexpr (KT > 0) {
                        const unsigned* rp = rows0 + (size_t)o * NW;
#pragma unroll
                        for (int i = 0; i < NW; ++i) w[u][i] = __ldg(rp + i);
                    }
                }
            }
            M dR[U];                 // accessed set of a deferred token
            unsigned drank[U];       // ranks of its pending slots (0 = the token is not deferred)
            unsigned dmeta[U];
            bool dmulti[U];          // more than one pending slot
            int ndef = 0;            // this lane's deferred tokens of the batch: one pending slot | several << 16
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int o = ob + u * S;
                const bool live = (unsigned)f[u] < (unsigned)F;
                drank[u] = 0u;
                dmeta[u] = 0u;
                dmulti[u] = false;
                dR[u] = 0;
                if (live) {
                    unsigned a2[KM];            // byte offsets into the table (tab16 with replicas, else the byte table)
                    constexpr unsigned SC = REP ? 2u : 1u;      // bytes per table entry
                    if constexpr (KT > 0) {
#pragma unroll
                        for (int i = 0; i < NW; ++i) {
                            // both ids of the word at once: anything outside [0,512) becomes 512, the "not an expert"
                            // entry (unsigned 16-bit minimum: -1 = 0xffff, an empty slot, included)
                            const unsigned wc = __vminu2(w[u][i], 0x02000200u);
                            const unsigned ws = REP ? wc + wc : wc;     // ids <= 512: the doubling does not carry
                            a2[2 * i] = ws & 0xffffu;
                            a2[2 * i + 1] = ws >> 16;
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < 16; ++j)
                            a2[j] = (j < k) ? SC * min((unsigned)(unsigned short)__ldg(base + ((size_t)t0 + o) * k + j), 512u) : 512u * SC;
                    }
                    // all table lookups first, then no branch: a slot that is not a plain expert has row 64, which
                    // shifts to an empty mask and counts into the sink row.  Without replicas the byte table already
                    // holds the row: the partition, or kBadFlag = 64 = the sink.
                    unsigned t[KM];
#pragma unroll
                    for (int j = 0; j < KM; ++j) {
                        if constexpr (REP) t[j] = slds_u16(tb + a2[j]);
                        else t[j] = slds_u8(pb8 + a2[j]);
                    }
                    M R = 0;
                    unsigned ranks = 0u;
#pragma unroll
                    for (int j = 0; j < KM; ++j) {
                        const unsigned row = REP ? (t[j] >> 7) : t[j];
                        TACG_ASSERT(a2[j] <= 512u * SC && (row < (unsigned)P || row == (unsigned)kSink));
                        R |= bit_or_zero<M>(row);
                        if constexpr (REP) sred_inc((t[j] & 0x3f80u) | cl);      // the row field is the byte offset of the row
                        else sred_inc(cl + row * 128u);
                        if (RECS && j < 8) ranks |= (t[j] & 15u) << (4 * j);
                    }
                    if constexpr (OUT) {
                        if (serve_l) {
                            signed char* out = serve_l + (size_t)o * k;
#pragma unroll
                            for (int j = 0; j < KM; ++j)
                                if (j < k) out[j] = ((REP ? (t[j] & kT16Bad) : (t[j] & kBadFlag)) != 0u) ? (signed char)-1 : (signed char)((REP ? t[j] >> 7 : t[j]) & 0x3fu);
                        }
                    }
                    unsigned packed = 1u << 22;          // one token of family f
                    if (!RECS || ranks == 0u) {
                        const int nR = popc_m<M>(R), rem = popc_m<M>(R & ~((M)1 << home));
                        packed |= (unsigned)max(0, nR - 1) | ((unsigned)rem << 11);
                        if (OUT && cost_l) cost_l[o] = (unsigned char)rem;
                    } else {
                        dR[u] = R;
                        drank[u] = ranks;
                        dmeta[u] = (unsigned)o | ((unsigned)f[u] << kOffBits) | ((unsigned)home << (kOffBits + 3));
                        const unsigned nz = (ranks | (ranks >> 1) | (ranks >> 2) | (ranks >> 3)) & 0x11111111u;
                        dmulti[u] = (nz & (nz - 1u)) != 0u;
                        ndef += dmulti[u] ? 0x10000 : 1;
                    }
                    sred_add(al + (unsigned)f[u] * 128u, packed);
                } else if (worker && o < n) {
                    if (OUT && cost_l) cost_l[o] = 0;
                    if (OUT && serve_l)
                        for (int j = 0; j < k; ++j) serve_l[(size_t)o * k + j] = -1;
                }
            }
            if constexpr (RECS) {
                // records of this batch: one warp-wide reservation (tokens with one pending slot | with several, 16 bits
                // each: an item has at most 32768 tokens), then every lane writes its own
                if (__any_sync(0xffffffffu, ndef != 0)) {
                    int inc = ndef;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        const int v = __shfl_up_sync(0xffffffffu, inc, d);
                        if (lane >= d) inc += v;
                    }
                    const int total = __shfl_sync(0xffffffffu, inc, 31);
                    unsigned wbase = 0u;
                    // (PTX directly: for atomicAdd under `if (lane == 31)` the compiler emits its generic warp-aggregation
                    // sequence, a vote, a leader election and a popcount, for an add that one lane executes)
                    if (lane == 31)
                        asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(wbase) : "r"(nrb), "r"((unsigned)total) : "memory");
                    wbase = __shfl_sync(0xffffffffu, wbase, 31);
                    const unsigned mine = wbase + (unsigned)(inc - ndef);
                    unsigned pos1 = mine & 0xffffu;                               // singles: upwards from entry 0
                    unsigned pos2 = (unsigned)g.slice - 1u - (mine >> 16);        // several: downwards from the last entry
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        if (drank[u]) {
                            const unsigned pos = dmulti[u] ? pos2-- : pos1++;
                            TACG_ASSERT(pos < (unsigned)g.slice && pos1 <= pos2 + 2u);
                            recs[pos] = make_rec<M>(dR[u], drank[u], dmeta[u]);
                        }
                    }
                }
            }
        }
        // item epilogue: per-family sums of this thread -> CTA, per-partition columns -> row
#pragma unroll
        for (int fq = 0; fq < 8; ++fq) {
            if (fq < F) {
                const unsigned av = acc[fq * 32];
                acc[fq * 32] = 0u;
                const unsigned s = __reduce_add_sync(0xffffffffu, av & 0x7ffu);
                const unsigned q = __reduce_add_sync(0xffffffffu, (av >> 11) & 0x7ffu);
                const unsigned c = __reduce_add_sync(0xffffffffu, av >> 22);
                if (lane == 0) {          // plain PTX: no compiler-generated warp aggregation around a one-lane add
                    if (s) sred_add(saddr(comm_s) + 4u * fq, s);
                    if (q) sred_add(saddr(comm_s) + 4u * (8 + fq), q);
                    if (c) sred_add(saddr(fam_s) + 4u * fq, c);
                }
            }
        }
        __syncthreads();
        unsigned* row = p.rows + (size_t)item * g.W;
        for (int m = tid >> 5; m < P; m += kEvalThreads / 32) {
            const unsigned s = __reduce_add_sync(0xffffffffu, cnt[m * 32 + lane]);
            cnt[m * 32 + lane] = 0u;
            if (lane == 0) row[m] = layer_ovf ? 0u : s;     // overflow: everything but the token counts is redone later
        }
        if (tid < F) {
            row[P + tid] = layer_ovf ? 0u : comm_s[tid];
            row[P + F + tid] = layer_ovf ? 0u : comm_s[8 + tid];
            row[P + 2 * F + tid] = fam_s[tid];
        }
        if (tid == 0) {
            row[P + 3 * F] = layer_ovf ? kOverflow : (nrec_s & 0xffffu);
            row[P + 3 * F + 1] = layer_ovf ? 0u : (nrec_s >> 16);
        }
        // next item
        hm0 += hstep;
        if (hm0 >= P) hm0 -= P;
        if (++sl == g.spm) {
            sl = 0;
            if (++mb == g.nmb) { mb = 0; ++layer; }
            hm0 = (int)((g.token_offset + mb * g.B) % P);
        }
    }
}

struct ChainParams {
    EvalGeom g;
    const int16_t* indices;
    const int8_t* family;
    const int8_t* primary;
    const int8_t* replicas;
    const unsigned* rows;
    const Rec* rec;
    float theta;
    double rho;
    double* load_state;                // [L,P] in/out or null
    unsigned long long* load;          // [L,P] out
    unsigned long long* comm_span;     // [L,F] out
    unsigned long long* comm_remote;   // [L,F] out
    unsigned long long* ntok;          // [F] out
    unsigned char* cost;
    signed char* serve;
    int groups;                        // clusters in the grid; cluster c owns layers c, c + groups, ...
    int gper;                          // kModeGrid: CTAs per layer
    unsigned* gsync;                   // kModeGrid: [L][kSyncWords] zeroed before the launch (see layer_barrier)
};

// How the CTAs of one layer exchange the dispatch counts of a micro-batch.
constexpr int kModeSingle = 0;    // one CTA per layer: nothing to exchange
constexpr int kModeCluster = 1;   // one thread-block cluster per layer: distributed shared memory + the cluster barrier
constexpr int kModeGrid = 2;      // few layers: more CTAs per layer than a cluster holds, launched cooperatively (all
                                  // resident); counts through global atomics, one arrival counter per layer
// per-layer words of ChainParams::gsync: one 64-bit word per (micro-batch parity, partition), each on its own 128-byte
// line: arrivals << 48 | cumulative dispatch count.  A CTA adds (1 << 48) | its count with ONE atomic; the thread that
// owns partition m polls that word until the arrivals reach gper * (rounds of this parity): count and flag are one word,
// so there is no fence, no separate arrival counter and no read-back.  Then sums u64[16] | arrivals of the layer's
// last barrier (layer_barrier).
constexpr int kSyncSums = 4096, kSyncBar = 4160, kSyncWords = 4224;

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* ptr) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ptr) : "memory");
    return v;
}

__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long* ptr) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(ptr) : "memory");
    return v;
}

// Barrier of the CTAs of one layer (kModeGrid; the launch is cooperative, so all of them are resident): the `n`-th
// call returns once gper * n arrivals are counted.  What the CTA's threads wrote or added before is visible to every
// CTA after.  A CTA that waits longer than seconds has met a bug, not a slow peer: it traps instead of hanging the GPU.
__device__ __forceinline__ void layer_barrier(unsigned* bar, unsigned target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(bar, 1u);
        const long long t0 = clock64();
        while (ld_acquire_u32(bar) < target)
            if (clock64() - t0 > (1ll << 33)) __trap();
        __threadfence();
    }
    __syncthreads();
}

// One cluster of CS CTAs per layer (MODE: kModeSingle a plain CTA, kModeGrid gper CTAs of a cooperative grid).  CTA `rank` takes the rank-th share of every
// item's records; the integer dispatch counts of a micro-batch are exchanged through distributed shared
// memory (two alternating buffers, one cluster barrier per micro-batch).
template <typename M, bool OUT, int MODE>
__global__ void __launch_bounds__(kChainThreads, MODE == kModeGrid ? 1 : 2) eval_chain_kernel(const ChainParams p) {
    tacg_pdl_prologue();
    extern __shared__ __align__(16) unsigned char csm[];
    const EvalGeom& g = p.g;
    const int P = g.P, E = g.E, F = g.F, r = g.r, k = g.k;
    LayerTables T;
    size_t off = 0;
    T.cand = csm + off;                                    off += ((size_t)E * kCandStride + 15) & ~(size_t)15;
    T.rep = reinterpret_cast<signed char*>(csm + off);     off += ((size_t)E * r + 15) & ~(size_t)15;
    unsigned* cnt = reinterpret_cast<unsigned*>(csm + off);   off += sizeof(unsigned) * (size_t)P * 32;
    // [warps][8][32] lane-private family words (span | remote << 16), not in grid mode (see finish below)
    unsigned* accb = reinterpret_cast<unsigned*>(csm + off);
    if (MODE != kModeGrid) off += sizeof(unsigned) * (kChainThreads / 32) * 8 * 32;
    unsigned short* replist = reinterpret_cast<unsigned short*>(csm + off);   // [E] ids of the replicated experts
    __shared__ unsigned char ptab_s[kPtab];
    __shared__ unsigned char rank8[kPtab];
    __shared__ __align__(16) unsigned char candr[(kMaxRank + 1) * kCandStride];   // candidate tables by rank
    __shared__ double Ls[64];                  // EMA state of this layer
    __shared__ unsigned long long Ks[64];      // order_key of Ls
    __shared__ unsigned long long ltot[64];    // cumulative integer load of this layer
    __shared__ unsigned long long csum[24];    // span | remote | tokens per family: rows of the scan kernel
    __shared__ unsigned long long dsum[16];    // span | remote of the deferred tokens handled by THIS CTA
    __shared__ unsigned dsum32[16];            // the same for the current round of slices: 32-bit shared atomics are native,
                                               // 64-bit ones are compare-and-swap loops that 16 warps contend on
    __shared__ unsigned exch[2][16][64];       // every cluster rank's dispatch counts of the micro-batch (even / odd):
                                               // each CTA stores its own row into all its peers before the barrier
    __shared__ unsigned wsum[kChainThreads / 32 + 1];
    __shared__ unsigned long long feas_s;
    __shared__ uint4 candfix[32];              // cand_fixed of the replicated experts of ranks 1..32
    __shared__ unsigned long long mine_s[64 + 24];   // the scan kernel's sums of the current micro-batch (row words)
    __shared__ __align__(16) unsigned long long candm[(kMaxRank + 1) * 4];   // by rank: one-hot masks (type M) of the first four candidates
    __shared__ unsigned bigq_s;                                 // ranks that list more than four candidates
    // record counts of up to 32 slices as prefix sums (one pending slot | several), and bit s = slice s of the round is
    // left to this kernel; two copies by micro-batch parity: the next micro-batch's are published during the current one
    __shared__ unsigned pre1[2][36], pre2[2][36];
    __shared__ unsigned ovf_s[2];
    T.ptab = ptab_s;
    T.S = Ls;                                  // the snapshot of a micro-batch IS the EMA state at its start

    const int tid = threadIdx.x, lane = tid & 31;
    int rank = 0, CS = 1;
    if constexpr (MODE == kModeCluster) {
        cg::cluster_group cgl = cg::this_cluster();
        rank = (int)cgl.block_rank();
        CS = (int)cgl.num_blocks();
    } else if constexpr (MODE == kModeGrid) {
        CS = p.gper;
        rank = (int)(blockIdx.x % (unsigned)CS);
    }
    const int cluster_id = blockIdx.x / CS;
    const unsigned cl = saddr_kept(cnt + lane);
    const unsigned db = saddr_kept(dsum32);
    unsigned* acc = accb + (tid >> 5) * (8 * 32) + lane;
    const unsigned al = saddr_kept(acc);
    const unsigned cmb = saddr_kept(candm), pbase1 = saddr(pre1), pbase2 = saddr(pre2);
    const int W = g.W;
    const int ncols = P + 3 * F;               // row words summed by threads 0..ncols-1

    for (int layer = cluster_id; layer < g.L; layer += p.groups) {
        __syncthreads();
        load_ptab(E, r, p.primary + (size_t)layer * E, p.replicas + (size_t)layer * E * r, T.ptab, T.rep);
        for (int i = tid; i < P * 32; i += kChainThreads) cnt[i] = 0u;
        if (tid < 64) {
            Ls[tid] = (p.load_state && tid < P) ? p.load_state[(size_t)layer * P + tid] : 0.0;
            Ks[tid] = order_key(Ls[tid]);
            ltot[tid] = 0ull;
        }
        if (tid < 24) csum[tid] = 0ull;
        if (tid < 16) { dsum[tid] = 0ull; dsum32[tid] = 0u; }
        if constexpr (MODE != kModeGrid) {
#pragma unroll
            for (int f = 0; f < 8; ++f) acc[f * 32] = 0u;
        }
        __syncthreads();
        const int nrep = build_ranks(E, T.ptab, rank8, replist, wsum);
        unsigned* gsl = MODE == kModeGrid ? p.gsync + (size_t)layer * kSyncWords : nullptr;
        unsigned long long gprev[2] = {0ull, 0ull};       // kModeGrid: the cumulative counts this thread read last, by parity
        unsigned nbar = 0u;                 // kModeGrid: barriers of this layer passed so far
        const int16_t* base = p.indices + (size_t)layer * (size_t)g.N * (size_t)k;
        const unsigned* rows_l = p.rows + (size_t)layer * g.ipl * W;
        const size_t rec_l = (size_t)layer * g.ipl * g.slice;

        // Per-family communication sums of a record.  Many records per thread and micro-batch (cluster, single CTA): one
        // conflict-free atomic into the thread's own word, span | remote << 16, folded once per round of slices
        // (flush_acc; 16-bit fields: a thread takes at most 32 * 32768 / 512 records of <= 16 each per round).  Few
        // records per thread (grid mode): two atomics straight into the CTA's words -- ATOMS.ADD does not merge lanes
        // that hit one word, so this costs several wavefronts per instruction, but there is no fold to pay for.
        auto add_comm = [&](unsigned fam, unsigned span, unsigned rem) {
            if constexpr (MODE == kModeGrid) {
                sred_add(db + fam * 4u, span);
                sred_add(db + 32u + fam * 4u, rem);
            } else {
                sred_add(al + fam * 128u, span | (rem << 16));
            }
        };
        auto flush_acc = [&]() {
            if constexpr (MODE != kModeGrid) {
#pragma unroll
                for (int fq = 0; fq < 8; ++fq) {
                    if (fq < F) {
                        const unsigned av = acc[fq * 32];
                        acc[fq * 32] = 0u;
                        const unsigned sp = __reduce_add_sync(0xffffffffu, av & 0xffffu);
                        const unsigned rq = __reduce_add_sync(0xffffffffu, av >> 16);
                        if (lane == 0) {
                            if (sp) sred_add(db + 4u * fq, sp);
                            if (rq) sred_add(db + 4u * (8 + fq), rq);
                        }
                    }
                }
            }
        };
        // a round of at most 32 slices adds less than 2^25 to a 32-bit sum; one thread per entry widens it between barriers
        auto fold_dsum = [&](int i) {
            dsum[i] += dsum32[i];
            dsum32[i] = 0u;
        };
        // record counts of up to 32 slices (one pending slot | several) and their prefix sums; one warp
        auto put_counts = [&](unsigned n1, unsigned n2, int ln, int buf) {
            const bool ovf = n1 == kOverflow;
            if (ovf) { n1 = 0u; n2 = 0u; }
            const unsigned om = __ballot_sync(0xffffffffu, ovf);
            if (ln == 0) ovf_s[buf] = om;
            unsigned a1 = n1, a2 = n2;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned v1 = __shfl_up_sync(0xffffffffu, a1, d), v2 = __shfl_up_sync(0xffffffffu, a2, d);
                if (ln >= d) { a1 += v1; a2 += v2; }
            }
            pre1[buf][ln + 1] = a1;
            pre2[buf][ln + 1] = a2;
            if (ln == 0) { pre1[buf][0] = 0u; pre2[buf][0] = 0u; }
        };
        auto load_counts = [&](const unsigned* rows_mb, int s0, int ns, int ln, int buf) {
            unsigned n1 = 0u, n2 = 0u;
            if (ln < ns) {
                n1 = rows_mb[(size_t)(s0 + ln) * W + ncols];
                n2 = rows_mb[(size_t)(s0 + ln) * W + ncols + 1];
            }
            put_counts(n1, n2, ln, buf);
        };
        // The second warp keeps the record counts of the first 32 slices of this micro-batch and the next in registers
        // (A, B) and has those of the one after in flight (C): nothing the chain waits for is a miss.
        const int ns0 = min(32, g.spm);
        auto fetch_counts = [&](long long mbx, unsigned& n1, unsigned& n2) {
            n1 = 0u;
            n2 = 0u;
            if (mbx < g.nmb && lane < ns0) {
                const unsigned* rn = rows_l + ((size_t)mbx * g.spm + lane) * W + ncols;
                n1 = rn[0];
                n2 = rn[1];
            }
        };
        auto prefetch_rows = [&](long long mb0, long long mb1) {      // rows of micro-batches [mb0, mb1) into L2
            mb1 = min(mb1, g.nmb);
            if (mb0 < mb1) {
                const unsigned* rp = rows_l + (size_t)mb0 * g.spm * W;
                const unsigned bytes = (unsigned)((mb1 - mb0) * g.spm * W * 4);
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(rp), "r"(bytes) : "memory");
            }
        };
        // step 3 for the replicated expert of rank i + 1: its candidates in the order of the snapshot
        auto cand_of = [&](int i, unsigned long long feas) {
            const int e = (int)replist[i];
            unsigned char* out = T.cand + e * kCandStride;
            if (r <= 3) {
                // at most four candidates: everything stays in registers between the order and the tables
                unsigned w0, w1;
                build_candidate_small(e, r, T, Ks, feas, w0, w1);
                unsigned* o = reinterpret_cast<unsigned*>(out);     // entries are 4-byte aligned (kCandStride = 12)
                o[0] = w0;
                o[1] = w1;
                if (i < kMaxRank) {
                    M* cm = reinterpret_cast<M*>(candm) + (i + 1) * 4;
                    cm[0] = (M)1 << ((w0 >> 8) & 0xffu);
                    cm[1] = (M)1 << ((w0 >> 16) & 0xffu);
                    cm[2] = (M)1 << (w0 >> 24);
                    cm[3] = (M)1 << (w1 & 0xffu);
                    unsigned* dst = reinterpret_cast<unsigned*>(candr + (i + 1) * kCandStride);
                    dst[0] = w0; dst[1] = w1; dst[2] = 0u;
                }
                return;
            }
            build_candidate(e, r, T, feas, out);
            if (i < kMaxRank) {
                // by rank: the one-hot masks of the first four candidates (entries beyond the count repeat the first)
                const int n = out[0];
                M* cm = reinterpret_cast<M*>(candm) + (i + 1) * 4;
#pragma unroll
                for (int q = 0; q < 4; ++q) cm[q] = (M)1 << out[1 + (q < n ? q : 0)];
                if (n > 4) atomicOr(&bigq_s, 1u << (i + 1));
                unsigned* dst = reinterpret_cast<unsigned*>(candr + (i + 1) * kCandStride);
                const unsigned* src = reinterpret_cast<const unsigned*>(out);
                dst[0] = src[0]; dst[1] = src[1]; dst[2] = src[2];
            }
        };
        // r <= 3 and at most 32 replicated experts (the usual case): lane i of the first warp owns the expert of rank i + 1
        const bool lane_owns = tid < nrep && nrep <= 32 && r <= 3;
        // (kept in shared memory, not in registers: the record loop of the other warps needs every register it has)
        if (lane_owns) {
            const CandFixed f0 = cand_fixed((int)replist[tid], r, T);
            candfix[tid] = make_uint4(f0.cpk, f0.okm, (unsigned)f0.cmask, (unsigned)(f0.cmask >> 32));
        }
        __syncwarp();
        auto put_tables = [&](int i, unsigned w0, unsigned w1) {
            unsigned* o = reinterpret_cast<unsigned*>(T.cand + (int)replist[i] * kCandStride);   // 4-byte aligned entries
            o[0] = w0;
            o[1] = w1;
            if (i < kMaxRank) {
                M* cm = reinterpret_cast<M*>(candm) + (i + 1) * 4;
                cm[0] = (M)1 << ((w0 >> 8) & 0xffu);
                cm[1] = (M)1 << ((w0 >> 16) & 0xffu);
                cm[2] = (M)1 << (w0 >> 24);
                cm[3] = (M)1 << (w1 & 0xffu);
                unsigned* dst = reinterpret_cast<unsigned*>(candr + (i + 1) * kCandStride);
                dst[0] = w0; dst[1] = w1; dst[2] = 0u;
            }
        };
        unsigned cA1 = 0u, cA2 = 0u, cB1 = 0u, cB2 = 0u;
        if (tid >= 32 && tid < 64) {
            if (lane == 0) prefetch_rows(0, 3);
            fetch_counts(0, cA1, cA2);
            fetch_counts(1, cB1, cB2);
            put_counts(cA1, cA2, lane, 0);
        }
        __syncthreads();
        for (long long mb = 0; mb < g.nmb; ++mb) {
            const unsigned* rows_mb = rows_l + (size_t)mb * g.spm * W;
            const int cur = (int)(mb & 1);                      // this micro-batch's copy of the record counts
            const unsigned pb1 = pbase1 + (unsigned)cur * 36u * 4u, pb2 = pbase2 + (unsigned)cur * 36u * 4u;
            // Grid mode: a thread has about one record per class and micro-batch, and the time of a micro-batch is a chain
            // of latencies.  The records do not depend on the snapshot: the first one of BOTH classes is located and its
            // load issued here, before the guard, so that the data is there when the candidate tables are.
            const unsigned first = (unsigned)rank * kChainThreads + tid;
            bool has1 = false, has2 = false;
            unsigned x1 = 0u, x2 = 0u;
            Rec v1 = {0u, 0u, 0u, 0u}, v2 = {0u, 0u, 0u, 0u};
            const unsigned slice0 = (unsigned)g.slice;
            auto locate0 = [&](unsigned pb, bool multi, unsigned gi) -> unsigned {
                unsigned sl = 0u, lo_sl = 0u, hi_sl = slds_u32(pb + 4u);
                while (gi >= hi_sl) {
                    ++sl;
                    lo_sl = hi_sl;
                    hi_sl = slds_u32(pb + 4u * (sl + 1u));
                }
                TACG_ASSERT(sl < (unsigned)ns0 && gi - lo_sl < slice0);
                return multi ? sl * slice0 + slice0 - 1u - (gi - lo_sl) : sl * slice0 + (gi - lo_sl);
            };
            auto early = [&]() {
                has1 = first < slds_u32(pb1 + 4u * ns0);
                has2 = first < slds_u32(pb2 + 4u * ns0);
                x1 = has1 ? locate0(pb1, false, first) : 0u;
                x2 = has2 ? locate0(pb2, true, first) : 0u;
                const Rec* recs0 = p.rec + rec_l + (size_t)mb * g.spm * (size_t)g.slice;
                v1 = recs0[x1];
                v2 = recs0[x2];
            };
            if constexpr (MODE == kModeGrid) {
                if (tid >= 32) early();       // the first warp has the guard to do first: its records follow the tables
            }
            // steps 1-2 by the first warp: guard of the snapshot (the EMA state: it only changes at the end of a
            // micro-batch).  The second warp meanwhile publishes this micro-batch's record counts.
            unsigned cC1 = 0u, cC2 = 0u;
            if (tid < 32) {
                // the order of an expert's candidates needs the loads only: its compares run under the guard's fp64 chain
                CandFixed cf = {0u, 0u, 0ull};
                if (lane_owns) {
                    const uint4 q = candfix[lane];
                    cf.cpk = q.x;
                    cf.okm = q.y;
                    cf.cmask = (unsigned long long)q.z | ((unsigned long long)q.w << 32);
                }
                const unsigned bef = lane_owns ? cand_order(cf.cpk, Ks) : 0u;
                const unsigned long long fm = load_guard_warp(Ls, P, p.theta, lane);
                if (lane == 0) { feas_s = fm; bigq_s = 0u; }
                __syncwarp();
                // step 3: the usual case, no second barrier
                if (lane_owns) {
                    unsigned w0, w1;
                    cand_tables(cf, bef, fm, w0, w1);
                    put_tables(lane, w0, w1);
                } else if (lane < nrep && nrep <= 32) cand_of(lane, fm);
                if constexpr (MODE == kModeGrid) early();
            } else if (tid < 64) {
                fetch_counts(mb + 2, cC1, cC2);
                if (lane == 0) prefetch_rows(mb + 3, mb + 4);
                put_counts(cB1, cB2, lane, cur ^ 1);      // the next micro-batch's counts: read after the barrier at its end
                // The records of the NEXT micro-batch do not depend on the chain: one bulk prefetch per slice and record
                // class pulls them into L2 now (a single instruction each, issued by one lane of one CTA per slice).
                if (mb + 1 < g.nmb && lane < ns0 && lane % CS == rank && cB1 != kOverflow) {
                    const Rec* rb = p.rec + rec_l + ((size_t)(mb + 1) * g.spm + lane) * (size_t)g.slice;
                    if (cB1) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(rb), "r"(cB1 * 16u) : "memory");
                    if (cB2) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(rb + (g.slice - cB2)), "r"(cB2 * 16u) : "memory");
                }
            } else if (tid >= 128 && tid < 128 + ncols) {
                // the scan kernel's sums of this micro-batch (independent of the chain; read again at step 5)
                unsigned long long mine = 0ull;
                for (int s = 0; s < g.spm; ++s) mine += rows_mb[(size_t)s * W + (tid - 128)];
                mine_s[tid - 128] = mine;
            }
            __syncthreads();
            // step 3 when the first warp could not take it
            if (nrep > 32) {
                const unsigned long long feas = feas_s;
                for (int i = tid; i < nrep; i += kChainThreads) cand_of(i, feas);
                __syncthreads();
            }
            const unsigned bigq = bigq_s;

            // one pending slot: rank q of the replicated expert, loc = accessed set so far | home; returns the pick:
            // the first of the (at most four) candidates in snapshot order that is local, else the first.  No branch.
            auto pick_slot = [&](unsigned q, M loc) -> M {
                M m1, m2, m3, m4;
                if constexpr (sizeof(M) == 4) {
                    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(m1), "=r"(m2), "=r"(m3), "=r"(m4) : "r"(cmb + q * 16u));
                } else {
                    asm volatile("ld.shared.v2.u64 {%0,%1}, [%2];" : "=l"(m1), "=l"(m2) : "r"(cmb + q * 32u));
                    asm volatile("ld.shared.v2.u64 {%0,%1}, [%2];" : "=l"(m3), "=l"(m4) : "r"(cmb + q * 32u + 16u));
                }
                M pm = m1;
                pm = (loc & m4) ? m4 : pm;
                pm = (loc & m3) ? m3 : pm;
                pm = (loc & m2) ? m2 : pm;
                pm = (loc & m1) ? m1 : pm;
                if (r > 3 && ((bigq >> q) & 1u) && !(loc & (m1 | m2 | m3 | m4)))     // more than four candidates listed
                    pm = (M)1 << pick_candidate<M>(candr + q * kCandStride, loc);
                return pm;
            };
            // step 4: the pending slots of this micro-batch.  The records of up to 32 slices form one index space per
            // record class, so that a thread's loads from different slices are in flight together.
            for (int s0 = 0; s0 < g.spm; s0 += 32) {
                const int ns = min(32, g.spm - s0);
                if (s0 > 0) {
                    __syncthreads();
                    if (tid < 32) load_counts(rows_mb, s0, ns, tid, cur);
                    else if (tid >= 96 && tid < 112) fold_dsum(tid - 96);
                    __syncthreads();
                }
                const size_t ro0 = rec_l + ((size_t)mb * g.spm + s0) * (size_t)g.slice;
                const Rec* recs = p.rec + ro0;
                const unsigned stride = (unsigned)CS * kChainThreads;
                const unsigned slice = (unsigned)g.slice;
                // per-token outputs of a record at entry x (OUT only): token index from the slice and the offset
                auto token_of = [&](unsigned x, unsigned meta) -> size_t {
                    long long t0, t1;
                    item_tokens(g, mb, s0 + (int)(x / slice), t0, t1);
                    return (size_t)layer * g.N + t0 + (meta & ((1u << kOffBits) - 1u));
                };
                // the pending slot whose rank sits at bit sh of the record's rank word
                auto step = [&](M& R, M hb, unsigned rk, int sh, unsigned meta, unsigned x) {
                    TACG_ASSERT(((rk >> sh) & 15u) >= 1u && (int)((rk >> sh) & 15u) <= nrep);
                    const M pm = pick_slot((rk >> sh) & 15u, R | hb);
                    R |= pm;
                    const int pick = sizeof(M) == 8 ? 63 - __clzll((long long)pm) : 31 - __clz((int)pm);
                    TACG_ASSERT(pick >= 0 && pick < P);
                    sred_inc(cl + (unsigned)pick * 128u);
                    if (OUT && p.serve) p.serve[token_of(x, meta) * k + (sh >> 2)] = (signed char)pick;
                };
                // one record: its pending slots in slot order (lowest nibble first), then the communication cost.
                // MULTI = false: the record class with exactly one pending slot, no loop.
                auto resolve = [&](auto MULTI, M R, unsigned rk, unsigned meta, unsigned x) {
                    const M hb = (M)1 << ((meta >> (kOffBits + 3)) & 63u);
                    if constexpr (decltype(MULTI)::value) {
                        while (rk) {
                            const int sh = (__ffs(rk) - 1) & ~3;
                            step(R, hb, rk, sh, meta, x);
                            rk &= ~(15u << sh);
                        }
                    } else {
                        step(R, hb, rk, (__ffs(rk) - 1) & ~3, meta, x);
                    }
                    const int nR = popc_m<M>(R), rem = popc_m<M>(R & ~hb);
                    if (OUT && p.cost) p.cost[token_of(x, meta)] = (unsigned char)rem;
                    add_comm((meta >> kOffBits) & 7u, (unsigned)max(0, nR - 1), (unsigned)rem);
                };
                // one record class: flat index gi over the slices' records of that class -> entry of the record array.
                // Within slice sl (flat indices [lo_sl, hi_sl)) the entry is xb + gi (first class, upwards from entry 0)
                // or xb - gi (second class, downwards from the last entry); a thread's indices only grow, and a whole
                // round of RF records usually stays inside one slice: one vote per round, no search.
                auto run_class = [&](auto MULTI, unsigned skip) {
                    constexpr unsigned RF = MODE == kModeGrid ? kRecFlightGrid : kRecFlight;
                    constexpr bool multi = decltype(MULTI)::value;
                    const unsigned pb = multi ? pb2 : pb1;               // shared address of the prefix sums
                    const unsigned tot = slds_u32(pb + 4u * ns);
                    unsigned sl = 0u, lo_sl = 0u, hi_sl = slds_u32(pb + 4u);
                    unsigned xb = multi ? slice - 1u : 0u;
                    auto advance = [&](unsigned gi) {
                        while (gi >= hi_sl) {
                            ++sl;
                            lo_sl = hi_sl;
                            hi_sl = slds_u32(pb + 4u * (sl + 1u));
                        }
                        TACG_ASSERT(sl < (unsigned)ns && gi - lo_sl < slice);
                        xb = multi ? sl * slice + slice - 1u + lo_sl : sl * slice - lo_sl;
                    };
                    const unsigned first = (unsigned)rank * kChainThreads + tid;
                    // the trip count is the warp's (lane 0 has the smallest index): the vote below is by the whole warp
                    for (unsigned g0 = first + skip * stride; g0 - lane < tot; g0 += RF * stride) {
                        // RF records per round, all their loads in flight before the first is used
                        unsigned x[RF];
                        Rec v[RF];
                        const unsigned glast = min(g0 + (RF - 1u) * stride, tot - 1u);
                        if (__any_sync(0xffffffffu, g0 < tot && glast >= hi_sl)) {
#pragma unroll
                            for (int q = 0; q < RF; ++q) {
                                const unsigned gq = g0 + (unsigned)q * stride;
                                x[q] = 0u;
                                if (gq < tot) {
                                    advance(gq);
                                    x[q] = multi ? xb - gq : xb + gq;
                                }
                            }
                        } else {
#pragma unroll
                            for (int q = 0; q < RF; ++q) {
                                const unsigned gq = g0 + (unsigned)q * stride;
                                x[q] = gq < tot ? (multi ? xb - gq : xb + gq) : 0u;
                            }
                        }
#pragma unroll
                        for (int q = 0; q < RF; ++q) v[q] = recs[x[q]];
                        if constexpr (!multi && !OUT && RF > 1) {
                            if (r <= 3) {
                                // One pending slot each and at most four candidates: straight-line code without a branch,
                                // so that the RF independent chains (shared load -> pick -> counter) overlap.  A record
                                // beyond the end stands in as rank 1 with its increments switched off.
                                M R[RF], hb[RF], pm[RF];
                                bool live[RF];
#pragma unroll
                                for (int q = 0; q < RF; ++q) {
                                    live[q] = g0 + (unsigned)q * stride < tot;
                                    const unsigned rk = live[q] ? v[q].z : 1u;
                                    const unsigned rq = (rk >> ((__ffs(rk) - 1) & ~3)) & 15u;
                                    R[q] = rec_set<M>(v[q]);
                                    hb[q] = (M)1 << ((v[q].w >> (kOffBits + 3)) & 63u);
                                    pm[q] = pick_slot(rq, R[q] | hb[q]);
                                }
#pragma unroll
                                for (int q = 0; q < RF; ++q) {
                                    R[q] |= pm[q];
                                    const int pick = sizeof(M) == 8 ? 63 - __clzll((long long)pm[q]) : 31 - __clz((int)pm[q]);
                                    const int nR = popc_m<M>(R[q]), rem = popc_m<M>(R[q] & ~hb[q]);
                                    if (live[q]) {
                                        sred_inc(cl + (unsigned)pick * 128u);
                                        add_comm((v[q].w >> kOffBits) & 7u, (unsigned)max(0, nR - 1), (unsigned)rem);
                                    }
                                }
                                continue;
                            }
                        }
                        if constexpr (multi && !OUT && RF > 1) {
                            if (r <= 3) {
                                // Several pending slots each: the RF records advance in lock step, one slot per pass, each
                                // pass straight-line code (RF independent chains); a record that is done, or beyond the
                                // end, stands in as rank 1 with its updates switched off.
                                M R[RF], hb[RF];
                                unsigned rk[RF], any = 0u;
                                bool live[RF];
#pragma unroll
                                for (int q = 0; q < RF; ++q) {
                                    live[q] = g0 + (unsigned)q * stride < tot;
                                    rk[q] = live[q] ? v[q].z : 0u;
                                    any |= rk[q];
                                    R[q] = rec_set<M>(v[q]);
                                    hb[q] = (M)1 << ((v[q].w >> (kOffBits + 3)) & 63u);
                                }
                                while (any) {
                                    M pm[RF];
                                    int sh[RF];
#pragma unroll
                                    for (int q = 0; q < RF; ++q) {
                                        const unsigned rkx = rk[q] ? rk[q] : 1u;
                                        sh[q] = (__ffs(rkx) - 1) & ~3;
                                        pm[q] = pick_slot((rkx >> sh[q]) & 15u, R[q] | hb[q]);
                                    }
                                    any = 0u;
#pragma unroll
                                    for (int q = 0; q < RF; ++q) {
                                        const int pick = sizeof(M) == 8 ? 63 - __clzll((long long)pm[q]) : 31 - __clz((int)pm[q]);
                                        if (rk[q]) {
                                            R[q] |= pm[q];
                                            sred_inc(cl + (unsigned)pick * 128u);
                                            rk[q] &= ~(15u << sh[q]);
                                        }
                                        any |= rk[q];
                                    }
                                }
#pragma unroll
                                for (int q = 0; q < RF; ++q) {
                                    const int nR = popc_m<M>(R[q]), rem = popc_m<M>(R[q] & ~hb[q]);
                                    if (live[q]) add_comm((v[q].w >> kOffBits) & 7u, (unsigned)max(0, nR - 1), (unsigned)rem);
                                }
                                continue;
                            }
                        }
#pragma unroll
                        for (int q = 0; q < RF; ++q)
                            if (g0 + (unsigned)q * stride < tot) resolve(MULTI, rec_set<M>(v[q]), v[q].z, v[q].w, x[q]);
                    }
                };
                if constexpr (MODE == kModeGrid) {
                    if (s0 == 0) {
                        // the two records loaded before the guard; what is left, if anything, goes through the loops
                        if (has1) resolve(std::false_type{}, rec_set<M>(v1), v1.z, v1.w, x1);
                        if (has2) resolve(std::true_type{}, rec_set<M>(v2), v2.z, v2.w, x2);
                    }
                    run_class(std::false_type{}, s0 == 0 ? 1u : 0u);
                    run_class(std::true_type{}, s0 == 0 ? 1u : 0u);
                } else {
                    run_class(std::false_type{}, 0u);
                    run_class(std::true_type{}, 0u);
                }
                // items left to this kernel: their tokens are served here, from the trace
                for (unsigned om = ovf_s[cur]; om; om &= om - 1u) {
                    const int s = s0 + __ffs(om) - 1;
                    long long t0, t1;
                    item_tokens(g, mb, s, t0, t1);
                    const unsigned hb0 = (unsigned)((g.token_offset + t0) % P);
                    const long long n = t1 - t0;
                    const long long lo = n * rank / CS, hi = n * (rank + 1) / CS;
                    for (long long o = lo + tid; o < hi; o += kChainThreads) {
                        const int fq = p.family[t0 + o];
                        if ((unsigned)fq >= (unsigned)F) continue;
                        int e[16], sv[16];
#pragma unroll
                        for (int j = 0; j < 16; ++j) e[j] = (j < k) ? (int)__ldg(base + ((size_t)t0 + o) * k + j) : -1;
                        const int home = (int)((hb0 + o) % P);
                        const M R = serve_token<16, M>(e, k, E, home, T, sv);
#pragma unroll
                        for (int j = 0; j < 16; ++j)
                            if (j < k && sv[j] >= 0) sred_inc(cl + (unsigned)sv[j] * 128u);
                        const int nR = popc_m<M>(R), rem = popc_m<M>(R & ~((M)1 << home));
                        if (OUT && p.cost) p.cost[(size_t)layer * g.N + t0 + o] = (unsigned char)rem;
                        if (OUT && p.serve)
                            for (int j = 0; j < k; ++j) p.serve[((size_t)layer * g.N + t0 + o) * k + j] = (signed char)sv[j];
                        add_comm((unsigned)fq, (unsigned)max(0, nR - 1), (unsigned)rem);
                    }
                }
                flush_acc();
            }
            // step 5: integer dispatch counts of the micro-batch, then Eq. 15
            __syncthreads();
            const int par = (int)(mb & 1);
            for (int m = tid >> 5; m < P; m += kChainThreads / 32) {
                const unsigned sm = __reduce_add_sync(0xffffffffu, cnt[m * 32 + lane]);
                cnt[m * 32 + lane] = 0u;
                if constexpr (MODE == kModeCluster) {
                    // lane q stores this CTA's count into rank q's table: after the barrier every CTA sums local words
                    if (lane < CS) cg::this_cluster().map_shared_rank(&exch[par][rank][m], lane)[0] = sm;
                } else if constexpr (MODE == kModeGrid) {
                    // cumulative per parity: nobody adds to this parity again before every CTA has passed the NEXT
                    // barrier, that is, after every CTA has read it
                    if (lane == 0)
                        atomicAdd(reinterpret_cast<unsigned long long*>(gsl + (par * 64 + m) * 32), (1ull << 48) | sm);
                } else {
                    if (lane == 0) exch[par][0][m] = sm;
                }
            }
            if constexpr (MODE == kModeCluster) cg::this_cluster().sync();
            else if constexpr (MODE != kModeGrid) __syncthreads();
            if (tid < P) {
                unsigned long long d = mine_s[tid];
                if constexpr (MODE == kModeGrid) {
                    // wait for the gper additions of this micro-batch to this partition's word
                    const unsigned long long* src = reinterpret_cast<const unsigned long long*>(gsl + (par * 64 + tid) * 32);
                    const unsigned want = ((unsigned)CS * (unsigned)((mb >> 1) + 1)) & 0xffffu;
                    unsigned long long now;
                    const long long t0 = clock64();
                    while ((short)((unsigned)((now = ld_relaxed_u64(src)) >> 48) - want) < 0)
                        if (clock64() - t0 > (1ll << 33)) __trap();          // a bug, not a slow peer: do not hang the GPU
                    now &= (1ull << 48) - 1ull;
                    d += now - gprev[par];
                    gprev[par] = now;
                } else {
                    for (int q = 0; q < CS; ++q) d += exch[par][q][tid];
                }
                const double ln = __dadd_rn(__dmul_rn(p.rho, Ls[tid]), (double)d);   // no FMA (Q19)
                Ls[tid] = ln;
                Ks[tid] = order_key(ln);
                ltot[tid] += d;
            } else if (tid < ncols) {
                csum[tid - P] += mine_s[tid];
            }
            if (tid >= 96 && tid < 112) fold_dsum(tid - 96);
            cA1 = cB1; cA2 = cB2;
            cB1 = cC1; cB2 = cC2;
            __syncthreads();
        }
        // layer epilogue: rank 0 adds the deferred tokens' communication sums of its peers and writes the outputs
        if constexpr (MODE == kModeCluster) cg::this_cluster().sync();
        if constexpr (MODE == kModeGrid) {
            if (tid < 16 && dsum[tid]) atomicAdd(reinterpret_cast<unsigned long long*>(gsl + kSyncSums) + tid, dsum[tid]);
            layer_barrier(gsl + kSyncBar, (unsigned)CS * ++nbar);
        }
        if (rank == 0) {
            if (tid < P) {
                p.load[(size_t)layer * P + tid] = ltot[tid];
                if (p.load_state) p.load_state[(size_t)layer * P + tid] = Ls[tid];
            } else if (tid >= 64 && tid < 64 + 2 * F) {
                const int which = (tid - 64) / F, f = (tid - 64) % F;
                unsigned long long v = csum[which * F + f];
                if constexpr (MODE == kModeCluster) {
                    cg::cluster_group cgl = cg::this_cluster();
                    for (int q = 0; q < CS; ++q) v += cgl.map_shared_rank(&dsum[0], q)[which * 8 + f];
                } else if constexpr (MODE == kModeGrid) {
                    v += __ldcg(reinterpret_cast<const unsigned long long*>(gsl + kSyncSums) + which * 8 + f);
                } else {
                    v += dsum[which * 8 + f];
                }
                (which ? p.comm_remote : p.comm_span)[(size_t)layer * F + f] = v;
            } else if (layer == 0 && tid >= 128 && tid < 128 + F) {
                p.ntok[tid - 128] = csum[2 * F + (tid - 128)];
            }
        }
        if constexpr (MODE == kModeCluster) cg::this_cluster().sync();     // peers keep their sums until rank 0 has read them
    }
}

// O11: (jain, maxvio, cv) per layer and for the loads summed over layers, fp64 -> fp32.
// One CTA per output row (row L = loads summed over layers), 64 x 16 threads: thread (m, q) adds the
// layers q, q+16, ... of partition m, so no thread walks more than L/16 dependent loads; the
// statistics are then computed by one thread from the P sums in the fixed order m = 0..P-1.
// rows != nullptr (the no-replica path): the scan kernel left one row of partial sums per item
// (loads | span | remote | tokens per family | -); row l < L adds the `ipl` rows of its layer, applies Eq. 15
// (one micro-batch: the same two fp64 operations the chain kernel applies) and writes load, load_state,
// comm_span, comm_remote and, from layer 0, ntok; row L sums the loads of all layers.
__global__ void __launch_bounds__(1024) fairness_kernel(unsigned long long* __restrict__ load, int L, int P,
                                                       float* __restrict__ out, const unsigned* __restrict__ rows,
                                                       long long ipl, int W, int F, double rho,
                                                       double* __restrict__ load_state,
                                                       unsigned long long* __restrict__ comm_span,
                                                       unsigned long long* __restrict__ comm_remote,
                                                       unsigned long long* __restrict__ ntok) {
    tacg_pdl_prologue();
    __shared__ unsigned long long part[16][64];
    __shared__ unsigned long long cpart[16][24];      // span | remote | tokens per family, F <= 8 each
    __shared__ double x[64];
    const int row = blockIdx.x;
    const int m = threadIdx.x & 63, q = threadIdx.x >> 6;
    unsigned long long v = 0, csum = 0;
    if (rows) {
        // thread (m, q) adds the item rows q, q+16, ...
        if (row < L) {
            const unsigned* rl = rows + (size_t)row * ipl * W;
            for (long long c = q; c < ipl; c += 16) {
                if (m < P) v += rl[(size_t)c * W + m];
                if (m < 3 * F) csum += rl[(size_t)c * W + P + m];
            }
        } else if (m < P) {
            for (long long i = q; i < (long long)L * ipl; i += 16) v += rows[(size_t)i * W + m];
        }
        if (m < 24) cpart[q][m] = csum;
    } else if (m < P) {
        if (row < L) { if (q == 0) v = load[(size_t)row * P + m]; }
        else for (int l = q; l < L; l += 16) v += load[(size_t)l * P + m];
    }
    part[q][m] = v;
    __syncthreads();
    if (q == 0) {
        unsigned long long t = 0;
#pragma unroll
        for (int z = 0; z < 16; ++z) t += part[z][m];
        x[m] = (double)t;
        if (rows && row < L && m < P) {
            load[(size_t)row * P + m] = t;
            if (load_state) {
                const double Ls = load_state[(size_t)row * P + m];
                load_state[(size_t)row * P + m] = __dadd_rn(__dmul_rn(rho, Ls), (double)t);   // no FMA (Q19)
            }
        }
    } else if (q == 1 && rows && row < L && m < 3 * F) {
        unsigned long long t = 0;
#pragma unroll
        for (int z = 0; z < 16; ++z) t += cpart[z][m];
        const int which = m / F, f = m - which * F;
        if (which == 0) comm_span[(size_t)row * F + f] = t;
        else if (which == 1) comm_remote[(size_t)row * F + f] = t;
        else if (row == 0) ntok[f] = t;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0, sq = 0.0, mx = 0.0;
        for (int z = 0; z < P; ++z) { tot += x[z]; sq += x[z] * x[z]; mx = fmax(mx, x[z]); }
        double jain = 1.0, maxvio = 0.0, cv = 0.0;
        if (tot != 0.0) {
            const double mean = tot / (double)P;
            double var = 0.0;
            for (int z = 0; z < P; ++z) var += (x[z] - mean) * (x[z] - mean);
            var /= (double)P;
            jain = (tot * tot) / ((double)P * sq);
            maxvio = (mx - mean) / mean;
            cv = sqrt(var) / mean;
        }
        out[(size_t)row * 3 + 0] = (float)jain;
        out[(size_t)row * 3 + 1] = (float)maxvio;
        out[(size_t)row * 3 + 2] = (float)cv;
    }
}

// The literal Eq. 15 (the load state decays after EVERY token) and any other short
// micro-batch: one warp per layer walks the micro-batches in order, lanes over the tokens of a micro-batch,
// the whole state in the warp's shared memory.  No other warp is ever waited for, so a trace of a million
// tokens per layer at B = 1 is a second of work instead of a million grid barriers.
struct SeqParams {
    EvalGeom g;
    const int16_t* indices;
    const int8_t* family;
    const int8_t* primary;
    const int8_t* replicas;
    float theta;
    double rho;
    double* load_state;
    unsigned long long* load;
    unsigned long long* comm_span;
    unsigned long long* comm_remote;
    unsigned long long* ntok;
    unsigned char* cost;
    signed char* serve;
};

template <typename M>
__global__ void __launch_bounds__(32) eval_seq_kernel(const SeqParams p) {
    tacg_pdl_prologue();
    extern __shared__ __align__(16) unsigned char qsm[];
    const EvalGeom& g = p.g;
    const int P = g.P, E = g.E, F = g.F, r = g.r, k = g.k;
    LayerTables T;
    size_t off = 0;
    T.S = reinterpret_cast<double*>(qsm + off);            off += 64 * sizeof(double);
    double* Ls = reinterpret_cast<double*>(qsm + off);     off += 64 * sizeof(double);
    unsigned long long* ltot = reinterpret_cast<unsigned long long*>(qsm + off);   off += 64 * sizeof(unsigned long long);
    unsigned long long* comm = reinterpret_cast<unsigned long long*>(qsm + off);   off += 24 * sizeof(unsigned long long);
    unsigned* cnt = reinterpret_cast<unsigned*>(qsm + off);                         off += 64 * sizeof(unsigned);
    unsigned short* replist = reinterpret_cast<unsigned short*>(qsm + off);         off += ((size_t)E * 2 + 15) & ~(size_t)15;
    T.ptab = qsm + off;                                    off += kPtab + 12;
    T.cand = qsm + off;                                    off += ((size_t)E * kCandStride + 15) & ~(size_t)15;
    T.rep = reinterpret_cast<signed char*>(qsm + off);
    __shared__ unsigned long long feas_s;
    __shared__ int nrep_s;
    const int lane = threadIdx.x;
    const int layer = blockIdx.x;
    load_ptab(E, r, p.primary + (size_t)layer * E, p.replicas + (size_t)layer * E * r, T.ptab, T.rep);
    for (int m = lane; m < 64; m += 32) {
        Ls[m] = (p.load_state && m < P) ? p.load_state[(size_t)layer * P + m] : 0.0;
        ltot[m] = 0ull;
        cnt[m] = 0u;
    }
    if (lane < 24) comm[lane] = 0ull;
    if (lane == 0) nrep_s = 0;
    __syncwarp();
    for (int e = lane; e < E; e += 32)
        if (T.ptab[e] & kRepFlag) replist[atomicAdd(&nrep_s, 1)] = (unsigned short)e;
    __syncwarp();
    const int nrep = nrep_s;
    const int16_t* base = p.indices + (size_t)layer * (size_t)g.N * (size_t)k;
    unsigned long long span[8] = {0, 0, 0, 0, 0, 0, 0, 0}, remote[8] = {0, 0, 0, 0, 0, 0, 0, 0}, seen[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (long long mb = 0; mb < g.nmb; ++mb) {
        // steps 1-3: snapshot, guard, candidate tables
        for (int m = lane; m < 64; m += 32) T.S[m] = Ls[m];
        __syncwarp();
        if (lane == 0) feas_s = load_guard(T.S, P, p.theta);
        __syncwarp();
        const unsigned long long feas = feas_s;
        for (int i = lane; i < nrep; i += 32) build_candidate((int)replist[i], r, T, feas, T.cand + (int)replist[i] * kCandStride);
        __syncwarp();
        // step 4: the tokens of the micro-batch, one per lane
        const long long t0 = mb * g.B, t1 = min(g.N, t0 + g.B);
        for (long long t = t0 + lane; t < t1; t += 32) {
            const int fq = p.family[t];
            if ((unsigned)fq >= (unsigned)F) {
                if (p.cost) p.cost[(size_t)layer * g.N + t] = 0;
                if (p.serve)
                    for (int j = 0; j < k; ++j) p.serve[((size_t)layer * g.N + t) * k + j] = -1;
                continue;
            }
            int e[16], sv[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) e[j] = (j < k) ? (int)__ldg(base + (size_t)t * k + j) : -1;
            const int home = (int)((g.token_offset + t) % P);
            const M R = serve_token<16, M>(e, k, E, home, T, sv);
#pragma unroll
            for (int j = 0; j < 16; ++j)
                if (j < k && sv[j] >= 0) atomicAdd(&cnt[sv[j]], 1u);
            const int nR = popc_m<M>(R), rem = popc_m<M>(R & ~((M)1 << home));
            if (p.cost) p.cost[(size_t)layer * g.N + t] = (unsigned char)rem;
            if (p.serve)
                for (int j = 0; j < k; ++j) p.serve[((size_t)layer * g.N + t) * k + j] = (signed char)sv[j];
#pragma unroll
            for (int q = 0; q < 8; ++q)
                if (q == fq) { span[q] += (unsigned)max(0, nR - 1); remote[q] += (unsigned)rem; seen[q] += 1; }
        }
        __syncwarp();
        // step 5: Eq. 15
        for (int m = lane; m < P; m += 32) {
            const unsigned d = cnt[m];
            cnt[m] = 0u;
            Ls[m] = __dadd_rn(__dmul_rn(p.rho, Ls[m]), (double)d);   // no FMA (Q19)
            ltot[m] += d;
        }
        __syncwarp();
    }
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        if (q < F) {
            atomicAdd(&comm[q], span[q]);
            atomicAdd(&comm[8 + q], remote[q]);
            atomicAdd(&comm[16 + q], seen[q]);
        }
    }
    __syncwarp();
    for (int m = lane; m < P; m += 32) {
        p.load[(size_t)layer * P + m] = ltot[m];
        if (p.load_state) p.load_state[(size_t)layer * P + m] = Ls[m];
    }
    if (lane < F) {
        p.comm_span[(size_t)layer * F + lane] = comm[lane];
        p.comm_remote[(size_t)layer * F + lane] = comm[8 + lane];
        if (layer == 0) p.ntok[lane] = comm[16 + lane];
    }
}

size_t select_smem_bytes(int E, int r) {
    return 64 * sizeof(double) + kPtab + (((size_t)E * kCandStride + 15) & ~(size_t)15) +
           (((size_t)E * (r > 0 ? r : 1) + 15) & ~(size_t)15);
}

// gesr_select: serve for one given snapshot; grid = (token blocks, layer)
template <int KT>
__global__ void __launch_bounds__(kEvalThreads)
select_kernel(const int16_t* __restrict__ indices, long long N, int k, int E, int P, int r,
              const int8_t* __restrict__ primary, const int8_t* __restrict__ replicas,
              const double* __restrict__ snapshot, float theta, long long token_offset, signed char* __restrict__ serve) {
    extern __shared__ __align__(16) unsigned char ssm[];
    constexpr int KM = KT > 0 ? KT : 16;
    LayerTables T;
    size_t off = 0;
    T.S = reinterpret_cast<double*>(ssm + off);            off += 64 * sizeof(double);
    T.ptab = ssm + off;                                    off += kPtab;
    T.cand = ssm + off;                                    off += ((size_t)E * kCandStride + 15) & ~(size_t)15;
    T.rep = reinterpret_cast<signed char*>(ssm + off);
    __shared__ unsigned long long feas_s;
    const int layer = blockIdx.y;
    load_ptab(E, replicas ? r : 0, primary + (size_t)layer * E, replicas ? replicas + (size_t)layer * E * r : nullptr,
              T.ptab, T.rep);
    if (threadIdx.x < 64) T.S[threadIdx.x] = threadIdx.x < P ? snapshot[(size_t)layer * P + threadIdx.x] : 0.0;
    __syncthreads();
    if (threadIdx.x == 0) feas_s = load_guard(T.S, P, theta);
    __syncthreads();
    build_candidates(E, replicas ? r : 0, T, feas_s);
    __syncthreads();
    const int16_t* base = indices + (size_t)layer * (size_t)N * (size_t)k;
    const long long stride = (long long)gridDim.x * kEvalThreads;
    for (long long t = (long long)blockIdx.x * kEvalThreads + threadIdx.x; t < N; t += stride) {
        int e[KM], sv[KM];
        tacg_load_ids<KT>(base + (size_t)t * k, k, e);
        const int home = (int)((token_offset + t) % P);
        serve_token<KM>(e, k, E, home, T, sv);
        signed char* out = serve + ((size_t)layer * N + t) * k;
        if constexpr (KT == 8) {
            int2 v;
            v.x = (sv[0] & 0xff) | ((sv[1] & 0xff) << 8) | ((sv[2] & 0xff) << 16) | ((sv[3] & 0xff) << 24);
            v.y = (sv[4] & 0xff) | ((sv[5] & 0xff) << 8) | ((sv[6] & 0xff) << 16) | ((sv[7] & 0xff) << 24);
            *reinterpret_cast<int2*>(out) = v;
        } else {
#pragma unroll
            for (int j = 0; j < KM; ++j)
                if (j < k) out[j] = (signed char)sv[j];
        }
    }
}

struct EvalCall {
    tacg_ctx* ctx;
    ScanParams sp;
    ChainParams cp;
    bool rep, out;
    int mode, cs, groups;      // chain_plan
};

template <int KT, bool REP, typename M, bool OUT>
int launch_scan(EvalCall& c) {
    tacg_ctx* ctx = c.ctx;
    auto kern = eval_scan_kernel<KT, REP, M, OUT>;
    const size_t smem = kCntAlign + sizeof(unsigned) * (kSink + 1) * 32 + sizeof(unsigned) * (kEvalThreads / 32) * 8 * 32;
    const long long T = (long long)c.sp.g.L * c.sp.g.ipl;
    const int grid = (int)max(1ll, min(T, (long long)ctx->sm_count * 2));
    TACG_CUDA_TRY(ctx, tacg_launch_pdl(kern, dim3(grid), dim3(kEvalThreads), smem, ctx->stream, c.sp));
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

// Tokens per scan item: the multiple of 512, at most kSlice, that gives the busiest CTA of the scan grid the least to do.
// A CTA takes ceil(items / CTAs) items; an item costs its tokens plus a fixed part, set to 2000 tokens' worth by
// measurement (the scan kernel's barriers and row sums, and what the chain kernel pays per slice: 400 gave three slices per
// micro-batch at config 4 and 2.82 ms, 2000 and more give two and 2.76 ms).  Large slices amortise the fixed part, small
// ones balance short traces.
static long long pick_slice(const tacg_ctx* ctx, int L, long long nmb, long long B) {
    const long long ctas = 2ll * ctx->sm_count;
    long long best = 512, best_cost = -1;
    // by the number of slices per micro-batch: the slices of a micro-batch are made as even as multiples of 512 allow
    for (long long spm = 1; spm <= (B + 511) / 512; ++spm) {
        const long long sl = ((B + spm - 1) / spm + 511) / 512 * 512;
        if (sl > kSlice) continue;
        const long long real_spm = (B + sl - 1) / sl;
        const long long items = (long long)L * nmb * real_spm;
        const long long per = (items + std::min(items, ctas) - 1) / std::min(items, ctas);
        const long long cost = per * ((B + real_spm - 1) / real_spm + 2000);
        if (best_cost < 0 || cost < best_cost) { best = sl; best_cost = cost; }
        if (sl <= 512) break;
    }
    return best;
}

// How the chain kernel is launched for a geometry: cluster size (or CTAs per layer of a cooperative grid) and mode.
void chain_plan(const tacg_ctx* ctx, const EvalGeom& g, int& mode, int& cs, int& groups) {
    // cluster size: as many CTAs per layer as the SM count allows, up to 16 (non-portable above 8)
    const int slots = 2 * ctx->sm_count;           // resident CTAs (two per SM)
    const long long tokens = std::min<long long>(g.B, g.N);
    // any size, not only powers of two: 5 at L = 58, 6 at L = 48; launch_chain lowers it if the clusters do not all fit
    cs = (int)std::max<long long>(1, std::min<long long>(16, slots / std::max(1, g.L)));
    if (cs > 8 && cs < 16) cs = 8;              // above the portable 8 only the full 16
    // a micro-batch with few records gains nothing from more CTAs
    cs = (int)std::max<long long>(1, std::min<long long>(cs, tokens / 2048));
    groups = std::min(g.L, std::max(1, slots / cs));
    mode = cs > 1 ? kModeCluster : kModeSingle;
    // few layers and long micro-batches: the largest cluster leaves most SMs idle.  One CTA per SM at most, about 1024
    // tokens of a micro-batch per CTA.
    if (cs == 16 && g.L * 32 <= ctx->sm_count && tokens >= 32 * 1024) {
        const int want = (int)std::min<long long>(ctx->sm_count / g.L, tokens / 1024);
        if (want > 16) {
            mode = kModeGrid;
            cs = want;
            groups = g.L;
        }
    }
}

template <typename M, bool OUT>
int launch_chain(EvalCall& c) {
    tacg_ctx* ctx = c.ctx;
    const EvalGeom& g = c.cp.g;
    const size_t smem = (((size_t)g.E * kCandStride + 15) & ~(size_t)15) +
                        (((size_t)g.E * g.r + 15) & ~(size_t)15) + sizeof(unsigned) * (size_t)g.P * 32 +
                        (c.mode != kModeGrid ? sizeof(unsigned) * (kChainThreads / 32) * 8 * 32 : 0) +
                        sizeof(unsigned short) * (size_t)g.E + 16;
    const int cs = c.cs;
    c.cp.groups = c.groups;
    c.cp.gper = cs;
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(c.cp.groups * cs);
    cfg.blockDim = dim3(kChainThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = ctx->stream;
    cudaLaunchAttribute attr[1];
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (c.mode == kModeGrid) {
        // every CTA of a layer waits for the others of that layer: cooperative, so the launch fails unless all fit
        attr[0].id = cudaLaunchAttributeCooperative;
        attr[0].val.cooperative = 1;
        auto kern = eval_chain_kernel<M, OUT, kModeGrid>;
        TACG_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        TACG_CUDA_TRY(ctx, cudaLaunchKernelEx(&cfg, kern, c.cp));
    } else if (c.mode == kModeCluster) {
        auto kern = eval_chain_kernel<M, OUT, kModeCluster>;
        TACG_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        if (cs > 8) TACG_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        // The clusters of all layers should be resident at once (a second wave would double the time): a cluster needs
        // its CTAs inside one GPC, so slots / cs over-estimates how many fit.  Ask the runtime, largest size first.
        // (the answer depends on the kernel, its shared memory, the device and L: remembered per process)
        static std::mutex memo_mutex;
        static std::map<std::tuple<const void*, size_t, int, int, int>, int> memo;
        const auto key = std::make_tuple((const void*)kern, smem, ctx->device, g.L, cs);
        int use = 0;
        {
            std::lock_guard<std::mutex> lock(memo_mutex);
            auto it = memo.find(key);
            if (it != memo.end()) use = it->second;
        }
        if (use == 0) {
            for (use = cs; use > 1; --use) {
                if (use > 8 && use < 16) continue;
                attr[0].val.clusterDim.x = use;
                cfg.gridDim = dim3(std::min(g.L, std::max(1, 2 * ctx->sm_count / use)) * use);
                int fit = 0;
                if (cudaOccupancyMaxActiveClusters(&fit, kern, &cfg) == cudaSuccess && fit * use >= (int)cfg.gridDim.x) break;
                (void)cudaGetLastError();
            }
            std::lock_guard<std::mutex> lock(memo_mutex);
            memo[key] = use;
        }
        if (use <= 1) {
            // not even pairs fit side by side: plain CTAs
            c.mode = kModeSingle;
            c.cs = 1;
            c.groups = std::min(g.L, 2 * ctx->sm_count);
            return launch_chain<M, OUT>(c);
        }
        c.cp.groups = std::min(g.L, std::max(1, 2 * ctx->sm_count / use));
        c.cp.gper = use;
        attr[0].val.clusterDim.x = use;
        cfg.gridDim = dim3(c.cp.groups * use);
        TACG_CUDA_TRY(ctx, cudaLaunchKernelEx(&cfg, kern, c.cp));
    } else {
        auto kern = eval_chain_kernel<M, OUT, kModeSingle>;
        TACG_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        cfg.numAttrs = 0;
        TACG_CUDA_TRY(ctx, cudaLaunchKernelEx(&cfg, kern, c.cp));
    }
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

template <int KT>
int launch_eval_t(EvalCall& c) {
    const bool wide = c.sp.g.P > 32;
    int rc;
    if (c.rep) {
        if (wide) rc = c.out ? launch_scan<KT, true, unsigned long long, true>(c) : launch_scan<KT, true, unsigned long long, false>(c);
        else rc = c.out ? launch_scan<KT, true, unsigned, true>(c) : launch_scan<KT, true, unsigned, false>(c);
        if (rc != TACG_OK) return rc;
        if (wide) return c.out ? launch_chain<unsigned long long, true>(c) : launch_chain<unsigned long long, false>(c);
        return c.out ? launch_chain<unsigned, true>(c) : launch_chain<unsigned, false>(c);
    }
    if (wide) rc = c.out ? launch_scan<KT, false, unsigned long long, true>(c) : launch_scan<KT, false, unsigned long long, false>(c);
    else rc = c.out ? launch_scan<KT, false, unsigned, true>(c) : launch_scan<KT, false, unsigned, false>(c);
    return rc;
}

template <int KT>
int launch_select_t(tacg_ctx* ctx, const int16_t* indices, int64_t N, int k, int L, int E, int P,
                    const int8_t* primary, const int8_t* replicas, int r, const double* snapshot, float theta,
                    int64_t token_offset, int8_t* serve) {
    const size_t smem = select_smem_bytes(E, r);
    const long long blocks = (N + kEvalThreads - 1) / kEvalThreads;
    const int gx = (int)max(1ll, min(blocks, (long long)max(1, ctx->sm_count * 8 / L)));
    select_kernel<KT><<<dim3(gx, L), kEvalThreads, smem, ctx->stream>>>(
        indices, (long long)N, k, E, P, r, primary, replicas, snapshot, theta, (long long)token_offset,
        reinterpret_cast<signed char*>(serve));
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

}  // namespace

int tacg_launch_select(tacg_ctx* ctx, const int16_t* indices, int64_t N, int k, int L, int E, int P,
                       const int8_t* primary, const int8_t* replicas, int r, const double* snapshot, float theta,
                       int64_t token_offset, int8_t* serve) {
    int kt = tacg_pick_kt(k, indices);
    if (kt == 8 && (reinterpret_cast<uintptr_t>(serve) % 8) != 0) kt = 0;
    switch (kt) {
        case 2: return launch_select_t<2>(ctx, indices, N, k, L, E, P, primary, replicas, r, snapshot, theta, token_offset, serve);
        case 4: return launch_select_t<4>(ctx, indices, N, k, L, E, P, primary, replicas, r, snapshot, theta, token_offset, serve);
        case 6: return launch_select_t<6>(ctx, indices, N, k, L, E, P, primary, replicas, r, snapshot, theta, token_offset, serve);
        case 8: return launch_select_t<8>(ctx, indices, N, k, L, E, P, primary, replicas, r, snapshot, theta, token_offset, serve);
        default: return launch_select_t<0>(ctx, indices, N, k, L, E, P, primary, replicas, r, snapshot, theta, token_offset, serve);
    }
}

int tacg_launch_eval(tacg_ctx* ctx, const int16_t* indices, const int8_t* family, int64_t N, int k, int L, int E,
                     int F, int P, const int8_t* primary, const int8_t* replicas, int r, float theta, double rho,
                     int64_t microbatch, int64_t token_offset, double* load_state, uint64_t* load,
                     uint64_t* comm_span, uint64_t* comm_remote, uint64_t* ntok, float* fairness,
                     uint8_t* cost_per_token, int8_t* serve) {
    if (N == 0) {
        TACG_CUDA_TRY(ctx, cudaMemsetAsync(comm_span, 0, sizeof(uint64_t) * (size_t)L * F, ctx->stream));
        TACG_CUDA_TRY(ctx, cudaMemsetAsync(comm_remote, 0, sizeof(uint64_t) * (size_t)L * F, ctx->stream));
        TACG_CUDA_TRY(ctx, cudaMemsetAsync(load, 0, sizeof(uint64_t) * (size_t)L * P, ctx->stream));
        TACG_CUDA_TRY(ctx, cudaMemsetAsync(ntok, 0, sizeof(uint64_t) * (size_t)F, ctx->stream));
    }
    const unsigned* fin_rows = nullptr;   // set when the fairness kernel still has the item rows to add
    long long fin_ipl = 0;
    int fin_W = 0;
    if (N > 0) {
        EvalCall c;
        c.ctx = ctx;
        c.rep = replicas != nullptr && r > 0;
        c.out = cost_per_token != nullptr || serve != nullptr;
        EvalGeom g;
        g.N = N; g.k = k; g.L = L; g.E = E; g.F = F; g.P = P; g.r = c.rep ? r : 0;
        g.B = (!c.rep || microbatch <= 0 || microbatch > N) ? N : microbatch;
        g.nmb = (N + g.B - 1) / g.B;
        g.k = k; g.token_offset = token_offset;
        if (c.rep && g.B < kSeqBelow) {
            // short micro-batches (down to the literal per-token Eq. 15): one warp per layer, nothing to exchange
            SeqParams q;
            g.spm = 1; g.slice = 512; g.ipl = g.nmb; g.W = 0;
            q.g = g;
            q.indices = indices; q.family = family; q.primary = primary; q.replicas = replicas;
            q.theta = theta; q.rho = rho; q.load_state = load_state;
            q.load = reinterpret_cast<unsigned long long*>(load);
            q.comm_span = reinterpret_cast<unsigned long long*>(comm_span);
            q.comm_remote = reinterpret_cast<unsigned long long*>(comm_remote);
            q.ntok = reinterpret_cast<unsigned long long*>(ntok);
            q.cost = cost_per_token;
            q.serve = reinterpret_cast<signed char*>(serve);
            const size_t smem = 64 * 8 * 3 + 24 * 8 + 64 * 4 + (((size_t)E * 2 + 15) & ~(size_t)15) + kPtab + 12 +
                                (((size_t)E * kCandStride + 15) & ~(size_t)15) + (((size_t)E * r + 15) & ~(size_t)15);
            tacg_prof_scope prof(ctx, TACG_PROF_EVAL);
            if (P > 32) {
                TACG_CUDA_TRY(ctx, cudaFuncSetAttribute(eval_seq_kernel<unsigned long long>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                TACG_CUDA_TRY(ctx, tacg_launch_pdl(eval_seq_kernel<unsigned long long>, dim3(L), dim3(32), smem, ctx->stream, q));
            } else {
                TACG_CUDA_TRY(ctx, cudaFuncSetAttribute(eval_seq_kernel<unsigned>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                TACG_CUDA_TRY(ctx, tacg_launch_pdl(eval_seq_kernel<unsigned>, dim3(L), dim3(32), smem, ctx->stream, q));
            }
            TACG_LAUNCH_CHECK(ctx);
        } else {
        const long long slice = pick_slice(ctx, L, g.nmb, g.B);
        g.slice = (int)slice;
        g.spm = (int)((g.B + slice - 1) / slice);
        g.ipl = g.nmb * g.spm;
        g.W = (int)tacg_align_up((size_t)P + 3 * (size_t)F + 2, 4);
        g.token_offset = token_offset;
        const int kt = tacg_pick_kt(k, indices);
        const size_t items = (size_t)L * (size_t)g.ipl;
        const size_t nrec = (c.rep && kt > 0) ? items * (size_t)g.slice : 0;      // one record per token at most
        const size_t o_rec = tacg_align_up(items * g.W * sizeof(unsigned), 256);
        c.mode = kModeSingle; c.cs = 1; c.groups = 1;
        if (c.rep) chain_plan(ctx, g, c.mode, c.cs, c.groups);
        const size_t o_sync = tacg_align_up(o_rec + nrec * sizeof(Rec), 256);
        const size_t total = o_sync + (c.mode == kModeGrid ? (size_t)L * kSyncWords * sizeof(unsigned) : 0);
        char* sbase = static_cast<char*>(tacg_scratch(ctx, total));
        if (!sbase) return TACG_ERR_CUDA;
        c.cp.gsync = reinterpret_cast<unsigned*>(sbase + o_sync);
        if (c.mode == kModeGrid)
            TACG_CUDA_TRY(ctx, cudaMemsetAsync(c.cp.gsync, 0, (size_t)L * kSyncWords * sizeof(unsigned), ctx->stream));
        c.sp.g = g;
        c.sp.indices = indices; c.sp.family = family; c.sp.primary = primary; c.sp.replicas = c.rep ? replicas : nullptr;
        c.sp.rows = reinterpret_cast<unsigned*>(sbase);
        c.sp.rec = reinterpret_cast<Rec*>(sbase + o_rec);
        c.sp.cost = cost_per_token;
        c.sp.serve = reinterpret_cast<signed char*>(serve);
        c.cp.g = g;
        c.cp.indices = indices; c.cp.family = family; c.cp.primary = primary; c.cp.replicas = replicas;
        c.cp.rows = c.sp.rows; c.cp.rec = c.sp.rec;
        c.cp.theta = theta; c.cp.rho = rho; c.cp.load_state = load_state;
        c.cp.load = reinterpret_cast<unsigned long long*>(load);
        c.cp.comm_span = reinterpret_cast<unsigned long long*>(comm_span);
        c.cp.comm_remote = reinterpret_cast<unsigned long long*>(comm_remote);
        c.cp.ntok = reinterpret_cast<unsigned long long*>(ntok);
        c.cp.cost = cost_per_token;
        c.cp.serve = reinterpret_cast<signed char*>(serve);
        c.cp.groups = 1; c.cp.gper = 1;
        int rc;
        {
            tacg_prof_scope prof(ctx, TACG_PROF_EVAL);
            switch (kt) {
                case 2: rc = launch_eval_t<2>(c); break;
                case 4: rc = launch_eval_t<4>(c); break;
                case 6: rc = launch_eval_t<6>(c); break;
                case 8: rc = launch_eval_t<8>(c); break;
                default: rc = launch_eval_t<0>(c); break;
            }
        }
        if (rc != TACG_OK) return rc;
        if (!c.rep) {
            fin_rows = c.sp.rows;
            fin_ipl = g.ipl;
            fin_W = g.W;
        }
        }
    }
    TACG_CUDA_TRY(ctx, tacg_launch_pdl(fairness_kernel, dim3(L + 1), dim3(1024), 0, ctx->stream,
                                       reinterpret_cast<unsigned long long*>(load), L, P, fairness, fin_rows, fin_ipl, fin_W,
                                       F, rho, load_state, reinterpret_cast<unsigned long long*>(comm_span),
                                       reinterpret_cast<unsigned long long*>(comm_remote),
                                       reinterpret_cast<unsigned long long*>(ntok)));
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// tacg_eval_primary_noalloc: the primary-only evaluation (no replica table: S8, S9, S11, S12 with every slot served by
// its primary partition) for callers that must not allocate -- code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc.  Same kernels, same geometry and therefore the same bits as tacg_eval_placement
// with replicas = NULL; the only difference is where the item rows of eval_scan_kernel live: not in the context's
// growable scratch (tacg_scratch: cudaMalloc / cudaFree) but in the fixed array below, which every GPU that loads the
// library holds until the process exits.
//
// The array's NAME is a host-side stand-in in host code, not a device address: the kernels are given the address that
// cudaGetSymbolAddress returns for the current device, looked up once per device (noalloc_rows).
// Every call shares the array and it keeps the last call's contents.  Nothing has to start at zero: eval_scan_kernel
// writes every word of every item row (loads | span | remote | tokens | two record counts) before fairness_kernel reads
// the first P + 3F of them.  Calls that overlap on the GPU (two streams, two contexts, two host threads on one
// device) race on it: the caller serialises them.
// ---------------------------------------------------------------------------------------------------------------------
namespace {

constexpr size_t kNoAllocBytes = TACG_NOALLOC_SCRATCH_BYTES;     // 8 MiB: config 4 whole (58 x 128 items of 48 words) fits many times
static __device__ __align__(256) unsigned char g_noalloc_rows[kNoAllocBytes];

constexpr int kMaxDevices = 64;
unsigned* g_noalloc_addr[kMaxDevices];       // device address of g_noalloc_rows on each device, 0 = not looked up yet
std::mutex g_noalloc_mutex;

// Device address of the array on ctx->device (which the caller has made current); looked up once per device.
int noalloc_rows(tacg_ctx* ctx, unsigned** out) {
    if (ctx->device < 0 || ctx->device >= kMaxDevices) {
        snprintf(ctx->detail, sizeof(ctx->detail), "eval_primary_noalloc: device ordinal %d not supported", ctx->device);
        return TACG_ERR_SHAPE;
    }
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_addr[ctx->device]) {
        void* ptr = nullptr;
        TACG_CUDA_TRY(ctx, cudaGetSymbolAddress(&ptr, g_noalloc_rows));
        if (!ptr || (reinterpret_cast<uintptr_t>(ptr) % 256) != 0) {
            snprintf(ctx->detail, sizeof(ctx->detail), "eval_primary_noalloc: bad symbol address %p", ptr);
            return TACG_ERR_CUDA;
        }
        g_noalloc_addr[ctx->device] = static_cast<unsigned*>(ptr);
    }
    *out = g_noalloc_addr[ctx->device];
    return TACG_OK;
}

template <int KT>
int launch_scan_primary(EvalCall& c) {
    const bool wide = c.sp.g.P > 32;
    if (wide) return c.out ? launch_scan<KT, false, unsigned long long, true>(c) : launch_scan<KT, false, unsigned long long, false>(c);
    return c.out ? launch_scan<KT, false, unsigned, true>(c) : launch_scan<KT, false, unsigned, false>(c);
}

}  // namespace

extern "C" int tacg_eval_primary_noalloc_prepare(tacg_ctx* ctx) {
    if (!ctx) return TACG_ERR_NULL;
    TACG_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    unsigned* rows = nullptr;
    return noalloc_rows(ctx, &rows);
}

extern "C" int tacg_eval_primary_noalloc(tacg_ctx* ctx, const int16_t* indices, const int8_t* family, int64_t N, int k,
                                         int L, int E, int F, int P, const int8_t* primary, double rho,
                                         int64_t token_offset, double* load_state, uint64_t* load, uint64_t* comm_span,
                                         uint64_t* comm_remote, uint64_t* ntok, float* fairness,
                                         uint8_t* cost_per_token, int8_t* serve) {
    if (!ctx) return TACG_ERR_NULL;
    if (N < 1 || k < 1 || k > 16 || L < 1 || E < 1 || E > 512 || F < 1 || F > 8 || P < 1 || P > 64 || token_offset < 0) {
        snprintf(ctx->detail, sizeof(ctx->detail), "eval_primary_noalloc: size out of range (N >= 1 here)");
        return TACG_ERR_SHAPE;
    }
    if (!indices || !family || !primary || !load || !comm_span || !comm_remote || !ntok || !fairness) {
        snprintf(ctx->detail, sizeof(ctx->detail), "eval_primary_noalloc: NULL pointer");
        return TACG_ERR_NULL;
    }
    TACG_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    // the geometry of tacg_launch_eval without replicas: one micro-batch, slices of at most kSlice tokens
    EvalCall c;
    c.ctx = ctx;
    c.rep = false;
    c.out = cost_per_token != nullptr || serve != nullptr;
    c.mode = kModeSingle; c.cs = 1; c.groups = 1;
    EvalGeom g;
    g.N = N; g.k = k; g.L = L; g.E = E; g.F = F; g.P = P; g.r = 0;
    g.B = N;
    g.nmb = 1;
    g.token_offset = token_offset;
    const long long slice = pick_slice(ctx, L, g.nmb, g.B);
    g.slice = (int)slice;
    g.spm = (int)((g.B + slice - 1) / slice);
    g.ipl = g.nmb * g.spm;
    g.W = (int)tacg_align_up((size_t)P + 3 * (size_t)F + 2, 4);
    const size_t need = (size_t)L * (size_t)g.ipl * (size_t)g.W * sizeof(unsigned);
    if (need > kNoAllocBytes) {
        snprintf(ctx->detail, sizeof(ctx->detail),
                 "eval_primary_noalloc: L * ceil(N / %d) * %d row words = %zu bytes of scratch, the fixed array holds %zu; "
                 "split the layers over several calls or use tacg_eval_placement",
                 g.slice, g.W, need, kNoAllocBytes);
        return TACG_ERR_SHAPE;
    }
    unsigned* rows = nullptr;
    int rc = noalloc_rows(ctx, &rows);
    if (rc != TACG_OK) return rc;
    memset(&c.sp, 0, sizeof(c.sp));
    c.sp.g = g;
    c.sp.indices = indices; c.sp.family = family; c.sp.primary = primary; c.sp.replicas = nullptr;
    c.sp.rows = rows;
    c.sp.rec = nullptr;
    c.sp.cost = cost_per_token;
    c.sp.serve = reinterpret_cast<signed char*>(serve);
    switch (tacg_pick_kt(k, indices)) {
        case 2: rc = launch_scan_primary<2>(c); break;
        case 4: rc = launch_scan_primary<4>(c); break;
        case 6: rc = launch_scan_primary<6>(c); break;
        case 8: rc = launch_scan_primary<8>(c); break;
        default: rc = launch_scan_primary<0>(c); break;
    }
    if (rc != TACG_OK) return rc;
    TACG_CUDA_TRY(ctx, tacg_launch_pdl(fairness_kernel, dim3(L + 1), dim3(1024), 0, ctx->stream,
                                       reinterpret_cast<unsigned long long*>(load), L, P, fairness,
                                       static_cast<const unsigned*>(rows), g.ipl, g.W, F, rho, load_state,
                                       reinterpret_cast<unsigned long long*>(comm_span),
                                       reinterpret_cast<unsigned long long*>(comm_remote),
                                       reinterpret_cast<unsigned long long*>(ntok)));
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

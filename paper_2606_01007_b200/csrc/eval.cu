// S8..S12: GESR serving selection (Eq. 13-14 + fallback), per-token
// communication cost (App. C), per-partition load, the decayed load state
// (Eq. 15, once per micro-batch per north_star / Q19) and fairness
// (Eq. 17-18).
//
// eval_kernel is persistent: the grid is split into groups of `cpl` CTAs, one group per
// layer (layers are independent problems, Q22).  Inside a layer the micro-batches are a
// serial chain: every CTA of the group adds its integer dispatch counts of micro-batch b to
// delta[l][b][:] in global memory, the group meets at a counter barrier, and each CTA then
// applies Eq. 15 redundantly from the same integers (same fp64 operations => the same bits),
// so no CTA ever reads another CTA's floating-point state.  The kernel is launched
// cooperatively whenever CTAs wait on one another.
//
// The pick rule of Q17 orders candidates by (not local, snapshot load, candidate slot).  Only the
// first key depends on the token, so once per micro-batch each replicated expert's feasible
// candidates are sorted by (snapshot load, slot) into a small table; a token then takes the first
// entry that is local to it (in its accessed set R or its home), else the first entry.  That is
// the same argmin, with all fp64 comparisons hoisted out of the token loop.
#include <cooperative_groups.h>

#include "tacg_common.cuh"

namespace {

constexpr int kEvalThreads = 512;
constexpr int kEvalBatch = 4;        // tokens per thread with their loads in flight together
constexpr int kCandStride = 12;      // bytes per expert in the candidate table: [0] = count, [1..9] = partitions
constexpr unsigned kRepFlag = 0x80u; // ptab bit: the expert has at least one replica
constexpr int kDeferCap = 64;        // deferred tokens per warp (at most 31 left over + 32 pushed)
constexpr int kDeferWords = 7;       // ids (<= 4 words), home | family << 8, token offset, pad; odd stride

struct LayerTables {
    unsigned char* ptab;   // [E] primary partition | kRepFlag
    unsigned char* cand;   // [E][kCandStride] sorted feasible candidates of replicated experts
    signed char* rep;      // [E*r] replica partitions as given, -1 = none
    double* S;             // [64] load snapshot
};

__device__ __forceinline__ void load_tables(int E, int r, const int8_t* __restrict__ pr,
                                            const int8_t* __restrict__ rp, const LayerTables& T) {
    for (int e = threadIdx.x; e < E; e += blockDim.x) {
        unsigned n = 0;
        for (int a = 0; a < r; ++a) {
            const signed char c = rp[(size_t)e * r + a];
            T.rep[e * r + a] = c;
            n += (c >= 0) ? 1u : 0u;
        }
        T.ptab[e] = (unsigned char)(((unsigned)pr[e] & 63u) | (n ? kRepFlag : 0u));
    }
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

// Candidate table of one snapshot: for every replicated expert the candidates (primary, then
// replicas in slot order), restricted to the feasible ones unless none is (fallback,
// PAPER.md:155), stably sorted by snapshot load (strict <, so ties keep slot order).
__device__ __forceinline__ void build_candidates(int E, int r, const LayerTables& T, unsigned long long feas) {
    for (int e = threadIdx.x; e < E; e += blockDim.x) {
        const unsigned in = T.ptab[e];
        if (!(in & kRepFlag)) continue;
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
        unsigned char* out = T.cand + e * kCandStride;
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
    }
}

// Pass 2 of the selection: replicated experts (bits of `pending`) in slot order; each takes the first
// local candidate of its sorted table, else the first, and joins R.
template <int KM, typename M>
__device__ __forceinline__ M serve_pending(const int (&e)[KM], unsigned pending, int home, M R, const LayerTables& T,
                                           int (&sv)[KM]) {
    const M hb = (M)1 << home;
    if constexpr (KM <= 8) {
        // Each lane walks its own set bits (lowest first = slot order), so a warp runs for the
        // largest number of replicated slots any of its tokens has, not for all KM slots.
        unsigned long long picks = 0ull;
        unsigned todo = pending;
        while (todo) {
            const int j = __ffs(todo) - 1;
            todo &= todo - 1u;
            int ex = e[0];
#pragma unroll
            for (int q = 1; q < KM; ++q) ex = (j == q) ? e[q] : ex;
            const unsigned char* c = T.cand + ex * kCandStride;
            const int n = c[0];
            int pick = c[1];
            const M loc = R | hb;
            for (int i = 1; i <= n; ++i) {
                const int v = c[i];
                if ((loc >> v) & (M)1) { pick = v; break; }
            }
            picks |= (unsigned long long)pick << (8 * j);
            R |= (M)1 << pick;
        }
#pragma unroll
        for (int j = 0; j < KM; ++j)
            if ((pending >> j) & 1u) sv[j] = (int)((picks >> (8 * j)) & 0xffull);
    } else {
#pragma unroll
        for (int j = 0; j < KM; ++j) {
            if (!((pending >> j) & 1u)) continue;
            const unsigned char* c = T.cand + e[j] * kCandStride;
            const int n = c[0];
            int pick = c[1];
            const M loc = R | hb;
            for (int i = 1; i <= n; ++i) {
                const int v = c[i];
                if ((loc >> v) & (M)1) { pick = v; break; }
            }
            sv[j] = pick;
            R |= (M)1 << pick;
        }
    }
    return R;
}

// Pass 2 on packed serve bytes (KM <= 8): svp byte j = serving partition of slot j.
template <int KM, typename M>
__device__ __forceinline__ M serve_pending_packed(const int (&e)[KM], unsigned pending, int home, M R,
                                                  const LayerTables& T, unsigned long long& svp) {
    const M hb = (M)1 << home;
    unsigned todo = pending;
    while (todo) {
        const int j = __ffs(todo) - 1;
        todo &= todo - 1u;
        int ex = e[0];
#pragma unroll
        for (int q = 1; q < KM; ++q) ex = (j == q) ? e[q] : ex;
        const unsigned char* c = T.cand + ex * kCandStride;
        const int n = c[0];
        int pick = c[1];
        const M loc = R | hb;
        for (int i = 1; i <= n; ++i) {
            const int v = c[i];
            if ((loc >> v) & (M)1) { pick = v; break; }
        }
        svp = (svp & ~(0xffull << (8 * j))) | ((unsigned long long)pick << (8 * j));
        R |= (M)1 << pick;
    }
    return R;
}

// All KM slots hold valid ids: pass 1 without branches.
template <int KM, bool REP, typename M>
__device__ __forceinline__ M serve_fast(const int (&e)[KM], int home, const LayerTables& T, int (&sv)[KM]) {
    M R = 0;
    unsigned pending = 0u;
#pragma unroll
    for (int j = 0; j < KM; ++j) {
        const unsigned in = T.ptab[e[j]];
        if constexpr (REP) {
            const unsigned isrep = in >> 7;
            sv[j] = (int)(in & 63u);
            R |= (M)(isrep ^ 1u) << (in & 63u);
            pending |= isrep << j;
        } else {
            sv[j] = (int)in;
            R |= (M)1 << in;
        }
    }
    if constexpr (REP) {
        if (pending) R = serve_pending<KM, M>(e, pending, home, R, T, sv);
    }
    return R;
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
    // pass 2: replicated experts in slot order; first local candidate of the sorted table, else the first
    if (pending) {
        R = serve_pending<KM, M>(e, pending, home, R, T, sv);
    }
    return R;
}

struct EvalParams {
    const int16_t* indices;
    const int8_t* family;
    long long N;
    int k, L, E, F, P, r;
    const int8_t* primary;
    const int8_t* replicas;
    float theta;
    double rho;
    long long B;            // micro-batch size (tokens)
    long long nmb;          // number of micro-batches
    long long token_offset;
    double* load_state;     // [L,P] in/out or null
    unsigned long long* load;          // [L,P] out
    unsigned long long* comm_span;     // [L,F] out (zeroed before launch, reduced atomically)
    unsigned long long* comm_remote;   // [L,F]
    unsigned long long* ntok;          // [F] out (zeroed before launch; counted by the CTAs of layer 0)
    unsigned char* cost;    // [L,N] or null
    signed char* serve;     // [L,N,k] or null
    unsigned long long* delta;   // scratch [L,nmb,P], zeroed before launch (only used when cpl > 1)
    unsigned* barrier;           // scratch [L], zeroed before launch
    unsigned long long* partial; // scratch [L,cpl,P+3F] (no-replica path): per-CTA loads | span | remote | tokens per family
    int cpl;                // CTAs per layer
    int groups;             // number of concurrent layer groups = gridDim.x / cpl
};

__host__ __device__ inline size_t eval_align16(size_t x) { return (x + 15) & ~(size_t)15; }

// carves the per-layer tables out of dynamic shared memory; returns the bytes used
__device__ __forceinline__ size_t carve_tables(unsigned char* base, int E, int r, LayerTables& T) {
    size_t off = 0;
    T.S = reinterpret_cast<double*>(base + off);            off += 64 * sizeof(double);
    T.ptab = base + off;                                    off += eval_align16((size_t)E);
    T.cand = base + off;                                    off += eval_align16((size_t)E * kCandStride);
    T.rep = reinterpret_cast<signed char*>(base + off);     off += eval_align16((size_t)E * (r > 0 ? r : 1));
    return off;
}

size_t tables_bytes(int E, int r) {
    return 64 * sizeof(double) + eval_align16((size_t)E) + eval_align16((size_t)E * kCandStride) +
           eval_align16((size_t)E * (r > 0 ? r : 1));
}

template <int KT>
__device__ __forceinline__ void unpack_ids(const unsigned (&w)[KT / 2], int (&e)[KT]) {
#pragma unroll
    for (int i = 0; i < KT / 2; ++i) {
        e[2 * i] = (int)(short)(w[i] & 0xffffu);
        e[2 * i + 1] = (int)w[i] >> 16;
    }
}

template <int KT>
__device__ __forceinline__ void load_row_raw(const int16_t* __restrict__ row, unsigned (&w)[KT / 2]) {
    if constexpr (KT == 8) {
        const uint4 v = __ldg(reinterpret_cast<const uint4*>(row));
        w[0] = v.x; w[1] = v.y; w[2] = v.z; w[3] = v.w;
    } else if constexpr (KT == 4) {
        const uint2 v = __ldg(reinterpret_cast<const uint2*>(row));
        w[0] = v.x; w[1] = v.y;
    } else {
#pragma unroll
        for (int i = 0; i < KT / 2; ++i) w[i] = __ldg(reinterpret_cast<const unsigned*>(row) + i);
    }
}

// KT: compile-time k (0 = generic), REP: a replica table is present, M: partition-set mask type
// (unsigned for P <= 32, else unsigned long long).
// OUT: per-token outputs (cost_per_token / serve) were requested.
template <int KT, bool REP, typename M, bool OUT>
__global__ void __launch_bounds__(kEvalThreads, 2)
eval_kernel(EvalParams p) {
    tacg_pdl_prologue();
    extern __shared__ __align__(16) unsigned char esm[];
    constexpr int KM = KT > 0 ? KT : 16;
    constexpr int U = KT > 0 ? kEvalBatch : 1;
    LayerTables T;
    size_t off = carve_tables(esm, p.E, p.r, T);
    unsigned long long* dsum = reinterpret_cast<unsigned long long*>(esm + off);   off += 64 * sizeof(unsigned long long);
    unsigned* cnt = reinterpret_cast<unsigned*>(esm + off);                        // [P][32], lane-private columns
    off += sizeof(unsigned) * (size_t)p.P * 32;
    // deferred-token queue of each warp (replicated slots are resolved 32 tokens at a time)
    constexpr bool kQueued = REP && KT > 0 && sizeof(M) == 4;
    unsigned* wqueue = reinterpret_cast<unsigned*>(esm + off) + (threadIdx.x >> 5) * (kDeferCap * kDeferWords);
    if (kQueued) off += sizeof(unsigned) * (size_t)(kEvalThreads / 32) * kDeferCap * kDeferWords;
    // per-family packed accumulators, one word per (warp, family, lane): a token is one shared atomic on its own
    // thread's word instead of a compare-select-add per family
    unsigned* acc = reinterpret_cast<unsigned*>(esm + off) + (threadIdx.x >> 5) * (8 * 32) + (threadIdx.x & 31);
    __shared__ double Ls[64];              // EMA state of this layer
    __shared__ unsigned long long ltot[64];  // cumulative integer load of this layer
    __shared__ unsigned long long feas_s;
    __shared__ unsigned long long comm_s[16];
    __shared__ unsigned fam_s[8];          // tokens per family seen by this CTA (layer 0 only)

    const int group = blockIdx.x / p.cpl;
    const int part = blockIdx.x % p.cpl;
    if (group >= p.groups) return;
    const int tid = threadIdx.x, lane = tid & 31;
    const int P = p.P, k = KT > 0 ? KT : p.k, E = p.E, F = p.F, r = REP ? p.r : 0;
    const int stepP = kEvalThreads % P;
    unsigned* cnt_lane = cnt + lane;

    for (int layer = group; layer < p.L; layer += p.groups) {
        __syncthreads();
        load_tables(E, r, p.primary + (size_t)layer * E, REP ? p.replicas + (size_t)layer * E * r : nullptr, T);
        for (int i = tid; i < P * 32; i += kEvalThreads) cnt[i] = 0u;
        if (tid < 64) {
            Ls[tid] = (p.load_state && tid < P) ? p.load_state[(size_t)layer * P + tid] : 0.0;
            ltot[tid] = 0ull;
        }
        if (tid < 16) comm_s[tid] = 0ull;
        if (tid < 8) fam_s[tid] = 0u;
        __syncthreads();
        // per family, over this thread's tokens: span (bits 0-10) | remote (11-21) | token count (22-31)
#pragma unroll
        for (int g = 0; g < 8; ++g) acc[g * 32] = 0u;
        int since = 0;                      // tokens added to acc since the last flush (uniform per warp)
        auto flush_acc = [&]() {
#pragma unroll
            for (int g = 0; g < 8; ++g) {
                if (g < F) {
                    const unsigned av = acc[g * 32];
                    const unsigned s = __reduce_add_sync(0xffffffffu, av & 0x7ffu);
                    const unsigned q = __reduce_add_sync(0xffffffffu, (av >> 11) & 0x7ffu);
                    if (lane == 0) {
                        if (s) atomicAdd(&comm_s[g], (unsigned long long)s);
                        if (q) atomicAdd(&comm_s[8 + g], (unsigned long long)q);
                    }
                    if (layer == 0) {               // tokens per family, counted once (family is shared by all layers)
                        const unsigned c = __reduce_add_sync(0xffffffffu, av >> 22);
                        if (lane == 0 && c) atomicAdd(&fam_s[g], c);
                    }
                    acc[g * 32] = 0u;
                }
            }
            since = 0;
        };
        const int16_t* base = p.indices + (size_t)layer * (size_t)p.N * (size_t)k;
        unsigned char* cost_l = (OUT && p.cost) ? p.cost + (size_t)layer * p.N : nullptr;
        signed char* serve_l = (OUT && p.serve) ? p.serve + (size_t)layer * p.N * k : nullptr;
        long long slice0 = 0;               // first token of the slice being processed (for the queued outputs)
        int qn = 0;                         // tokens waiting in this warp's queue (warp-uniform)
        // loads, communication cost and outputs of one token whose serve bytes are final; returns span | remote << 11 | 1 << 22
        auto finish_packed = [&](unsigned long long svp, M R, int hm, int o) -> unsigned {
#pragma unroll
            for (int j = 0; j < KM; ++j)
                if (j < 8) atomicAdd(cnt_lane + (unsigned)((svp >> (8 * j)) & 0xffull) * 32, 1u);
            const M notHome = ~((M)1 << hm);
            int nR, rem;
            if constexpr (sizeof(M) == 8) { nR = __popcll(R); rem = __popcll(R & notHome); }
            else { nR = __popc(R); rem = __popc(R & notHome); }
            if (OUT && cost_l) cost_l[slice0 + o] = (unsigned char)rem;
            if (OUT && serve_l) {
                signed char* out = serve_l + ((size_t)slice0 + o) * k;
#pragma unroll
                for (int j = 0; j < KM; ++j)
                    if (j < 8) out[j] = (signed char)((svp >> (8 * j)) & 0xffull);
            }
            return (unsigned)max(0, nR - 1) | ((unsigned)rem << 11) | (1u << 22);
        };
        // same for a token whose serving partitions are in registers (no replicated slot)
        auto finish_sv = [&](const int (&sv)[KM], M R, int hm, int o) -> unsigned {
#pragma unroll
            for (int j = 0; j < KM; ++j)
                if (j < k) atomicAdd(cnt_lane + sv[j] * 32, 1u);
            const M notHome = ~((M)1 << hm);
            int nR, rem;
            if constexpr (sizeof(M) == 8) { nR = __popcll(R); rem = __popcll(R & notHome); }
            else { nR = __popc(R); rem = __popc(R & notHome); }
            if (OUT && cost_l) cost_l[slice0 + o] = (unsigned char)rem;
            if (OUT && serve_l) {
                signed char* out = serve_l + ((size_t)slice0 + o) * k;
#pragma unroll
                for (int j = 0; j < KM; ++j)
                    if (j < k) out[j] = (signed char)sv[j];
            }
            return (unsigned)max(0, nR - 1) | ((unsigned)rem << 11) | (1u << 22);
        };
        // resolves the replicated slots of the last `nact` queued tokens, one token per lane
        auto drain = [&](int nact) {
            __syncwarp();
            if (lane < nact) {
                const unsigned* q = wqueue + (qn - nact + lane) * kDeferWords;
                unsigned ww[KT > 0 ? KT / 2 : 1];
#pragma unroll
                for (int i = 0; i < (KT > 0 ? KT / 2 : 1); ++i) ww[i] = q[i];
                int e[KM];
                if constexpr (KT > 0) unpack_ids<KT>(ww, e);
                const unsigned meta = q[4];
                const int hm = (int)(meta & 0xffu), fq = (int)(meta >> 8);
                unsigned long long svp = 0ull;
                unsigned pend = 0u;
                M R = 0;
                if constexpr (KM <= 8) {
#pragma unroll
                    for (int j = 0; j < KM; ++j) {          // pass 1 again, on packed serve bytes
                        const unsigned in = T.ptab[e[j]];
                        const unsigned isrep = in >> 7;
                        svp |= (unsigned long long)(in & 63u) << (8 * j);
                        R |= (M)(isrep ^ 1u) << (in & 63u);
                        pend |= isrep << j;
                    }
                    R = serve_pending_packed<KM, M>(e, pend, hm, R, T, svp);
                }
                const unsigned packed = finish_packed(svp, R, hm, (int)q[5]);
                atomicAdd(&acc[fq * 32], packed);         // queued tokens are live: fq < F
            }
            qn -= nact;
            __syncwarp();
        };

        for (long long mb = 0; mb < p.nmb; ++mb) {
            // steps 1-3: snapshot, guard, candidate tables
            if (REP) {
                if (tid < 64) T.S[tid] = Ls[tid];
                __syncthreads();
                if (tid == 0) feas_s = load_guard(T.S, P, p.theta);
                __syncthreads();
                build_candidates(E, r, T, feas_s);
                __syncthreads();
            }
            // step 4: this CTA's slice of the micro-batch
            const long long mb_begin = mb * p.B;
            const long long mb_end = min(p.N, mb_begin + p.B);
            const long long len = mb_end - mb_begin;
            const long long per = ((len + p.cpl - 1) / p.cpl + 31) / 32 * 32;
            const long long t0 = mb_begin + (long long)part * per;
            const long long t1 = min(mb_end, t0 + per);
            const int n = t1 > t0 ? (int)(t1 - t0) : 0;            // tokens of the slice (per <= 2^31 checked on the host)
            slice0 = t0;
            int home = (int)((p.token_offset + t0 + tid) % P);
            M notHome = ~((M)1 << home);            // constant over the slice when P divides the CTA width (stepP == 0)
            const int8_t* fam0 = p.family + t0;
            const unsigned* rows0 = reinterpret_cast<const unsigned*>(base + (size_t)t0 * k);   // KT > 0 only
            for (int ob = tid; ob < n + tid; ob += kEvalThreads * U) {      // uniform trip count across the CTA
                int f[U];
                unsigned w[U][KT > 0 ? KT / 2 : 1];
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const int o = ob + u * kEvalThreads;
                    f[u] = -1;
                    if (o < n) {
                        f[u] = fam0[o];
                        if constexpr (KT == 8) {
                            const uint4 v = __ldg(reinterpret_cast<const uint4*>(rows0) + o);
                            w[u][0] = v.x; w[u][1] = v.y; w[u][2] = v.z; w[u][3] = v.w;
                        } else if constexpr (KT == 4) {
                            const uint2 v = __ldg(reinterpret_cast<const uint2*>(rows0) + o);
                            w[u][0] = v.x; w[u][1] = v.y;
                        } else if constexpr (KT > 0) {
                            const unsigned* rp = rows0 + (size_t)o * (KT / 2);
#pragma unroll
                            for (int i = 0; i < KT / 2; ++i) w[u][i] = __ldg(rp + i);
                        }
                    }
                }
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const int o = ob + u * kEvalThreads;
                    const bool live = (unsigned)f[u] < (unsigned)F;
                    unsigned packed = 0;
                    bool defer = false;
                    unsigned pend = 0u;
                    if (live) {
                        int e[KM], sv[KM];
                        M R;
                        bool fast = false;
                        if constexpr (KT > 0) {
                            unpack_ids<KT>(w[u], e);
                            unsigned hi = (unsigned)e[0];       // a negative id is a huge unsigned value
#pragma unroll
                            for (int j = 1; j < KT; ++j) hi = max(hi, (unsigned)e[j]);
                            fast = hi < (unsigned)E;
                        } else {
#pragma unroll
                            for (int j = 0; j < 16; ++j)
                                e[j] = (j < k) ? (int)__ldg(base + ((size_t)t0 + o) * k + j) : -1;
                        }
                        bool done = true;
                        if constexpr (kQueued) {
                            if (fast) {
                                // pass 1; a token with replicated slots waits in the warp's queue (only its ids are kept)
                                M R1 = 0;
#pragma unroll
                                for (int j = 0; j < KM; ++j) {
                                    const unsigned in = T.ptab[e[j]];
                                    const unsigned isrep = in >> 7;
                                    sv[j] = (int)(in & 63u);
                                    R1 |= (M)(isrep ^ 1u) << (in & 63u);
                                    pend |= isrep;
                                }
                                defer = pend != 0u;
                                done = false;
                                if (!defer) packed = finish_sv(sv, R1, home, o);
                            }
                        }
                        if (done) {
                            if (fast) {
                                R = serve_fast<KM, REP, M>(e, home, T, sv);
#pragma unroll
                                for (int j = 0; j < KM; ++j) atomicAdd(cnt_lane + sv[j] * 32, 1u);
                            } else {
                                R = serve_token<KM, M>(e, k, E, home, T, sv);
#pragma unroll
                                for (int j = 0; j < KM; ++j)
                                    if (j < k && sv[j] >= 0) atomicAdd(cnt_lane + sv[j] * 32, 1u);
                            }
                            int nR, rem;
                            if constexpr (sizeof(M) == 8) { nR = __popcll(R); rem = __popcll(R & notHome); }
                            else { nR = __popc(R); rem = __popc(R & notHome); }
                            packed = (unsigned)max(0, nR - 1) | ((unsigned)rem << 11) | (1u << 22);
                            if (OUT && cost_l) cost_l[t0 + o] = (unsigned char)rem;
                            if (OUT && serve_l) {
                                signed char* out = serve_l + ((size_t)t0 + o) * k;
#pragma unroll
                                for (int j = 0; j < KM; ++j)
                                    if (j < k) out[j] = (signed char)sv[j];
                            }
                        }
                    } else if (o < n) {
                        if (OUT && cost_l) cost_l[t0 + o] = 0;
                        if (OUT && serve_l)
                            for (int j = 0; j < k; ++j) serve_l[((size_t)t0 + o) * k + j] = -1;
                    }
                    // packed is 0 unless f[u] is a family < F
                    if (packed) atomicAdd(&acc[f[u] * 32], packed);
                    if constexpr (kQueued) {
                        const unsigned dm = __ballot_sync(0xffffffffu, defer);
                        if (defer) {
                            unsigned* q = wqueue + (qn + __popc(dm & ((1u << lane) - 1u))) * kDeferWords;
#pragma unroll
                            for (int i = 0; i < KT / 2; ++i) q[i] = w[u][i];
                            q[4] = (unsigned)home | ((unsigned)f[u] << 8);
                            q[5] = (unsigned)o;
                        }
                        qn += __popc(dm);
                        if (qn >= 32) drain(32);
                    }
                    if (stepP) {
                        home += stepP;
                        if (home >= P) home -= P;
                        notHome = ~((M)1 << home);
                    }
                }
                since += kQueued ? 2 * U : U;     // a queued token adds to acc when it is drained
                if (since >= 120) flush_acc();      // 11-bit fields: 124 tokens x (span <= 15, remote <= 16) fit
            }
            if constexpr (kQueued) {
                while (qn > 0) drain(min(qn, 32));
            }
            flush_acc();
            // step 5: integer dispatch counts of the micro-batch, then Eq. 15
            __syncthreads();
            for (int m = tid >> 5; m < P; m += kEvalThreads / 32) {
                const unsigned s = __reduce_add_sync(0xffffffffu, cnt[m * 32 + lane]);
                cnt[m * 32 + lane] = 0u;
                if (lane == 0) dsum[m] = (unsigned long long)s;
            }
            __syncthreads();
            // Without replicas nothing depends on the snapshot (and the whole trace is one micro-batch): a CTA only
            // writes its own row of partial sums, never waits and never touches an accumulated output;
            // fairness_kernel adds the rows of a layer and applies Eq. 15.
            const bool ema_here = REP;
            if constexpr (REP) {
                if (p.cpl > 1) {
                    unsigned long long* dl = p.delta + ((size_t)layer * p.nmb + mb) * P;
                    if (tid < P && dsum[tid]) atomicAdd(&dl[tid], dsum[tid]);
                    __threadfence();
                    __syncthreads();
                    if (tid == 0) {
                        atomicAdd(&p.barrier[layer], 1u);
                        const unsigned target = (unsigned)((mb + 1) * p.cpl);
                        volatile unsigned* bar = p.barrier + layer;
                        while (*bar < target) __nanosleep(20);
                        __threadfence();
                    }
                    __syncthreads();
                    if (tid < P) dsum[tid] = __ldcg(&dl[tid]);
                    __syncthreads();
                }
            } else {
                if (tid < P) ltot[tid] += dsum[tid];
            }
            if (ema_here && tid < P) {
                const unsigned long long d = dsum[tid];
                Ls[tid] = __dadd_rn(__dmul_rn(p.rho, Ls[tid]), (double)d);   // no FMA (Q19)
                ltot[tid] += d;
            }
            __syncthreads();
        }
        // layer epilogue: communication sums and, from part 0, loads and the final state
        if constexpr (REP) {
            if (layer == 0 && tid < F && fam_s[tid]) atomicAdd(&p.ntok[tid], (unsigned long long)fam_s[tid]);
            if (tid < F) {
                if (comm_s[tid]) atomicAdd(&p.comm_span[(size_t)layer * F + tid], comm_s[tid]);
                if (comm_s[8 + tid]) atomicAdd(&p.comm_remote[(size_t)layer * F + tid], comm_s[8 + tid]);
            }
            if (part == 0 && tid < P) {
                p.load[(size_t)layer * P + tid] = ltot[tid];
                if (p.load_state) p.load_state[(size_t)layer * P + tid] = Ls[tid];
            }
        } else {
            unsigned long long* row = p.partial + ((size_t)layer * p.cpl + part) * (size_t)(P + 3 * F);
            if (tid < P) row[tid] = ltot[tid];
            if (tid < F) {
                row[P + tid] = comm_s[tid];
                row[P + F + tid] = comm_s[8 + tid];
                row[P + 2 * F + tid] = layer == 0 ? (unsigned long long)fam_s[tid] : 0ull;
            }
        }
    }
}

// O11: (jain, maxvio, cv) per layer and for the loads summed over layers, fp64 -> fp32.
// One CTA per output row (row L = loads summed over layers), 64 x 16 threads: thread (m, q) adds the
// layers q, q+16, ... of partition m, so no thread walks more than L/16 dependent loads; the
// statistics are then computed by one thread from the P sums in the fixed order m = 0..P-1.
// partial != nullptr (the no-replica path): the CTAs of the evaluation kernel left one row of partial sums each
// (loads | span | remote | tokens per family); row l < L adds the rows of its layer, applies Eq. 15 (one
// micro-batch: the same two fp64 operations the evaluation kernel applies) and writes load, load_state, comm_span,
// comm_remote and, from layer 0, ntok; row L sums the loads of all layers.
__global__ void __launch_bounds__(1024) fairness_kernel(unsigned long long* __restrict__ load, int L, int P,
                                                       float* __restrict__ out, const unsigned long long* __restrict__ partial,
                                                       int cpl, int F, double rho, double* __restrict__ load_state,
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
    if (partial) {
        // thread (m, q) adds the CTA rows q, q+16, ...: no thread walks more than cpl/16 dependent loads
        const size_t W = (size_t)(P + 3 * F);
        if (row < L) {
            const unsigned long long* rows = partial + (size_t)row * cpl * W;
            for (int c = q; c < cpl; c += 16) {
                if (m < P) v += rows[(size_t)c * W + m];
                if (m < 3 * F) csum += rows[(size_t)c * W + P + m];
            }
        } else if (m < P) {
            for (long long i = q; i < (long long)L * cpl; i += 16) v += partial[(size_t)i * W + m];
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
        if (partial && row < L && m < P) {
            load[(size_t)row * P + m] = t;
            if (load_state) {
                const double Ls = load_state[(size_t)row * P + m];
                load_state[(size_t)row * P + m] = __dadd_rn(__dmul_rn(rho, Ls), (double)t);   // no FMA (Q19)
            }
        }
    } else if (q == 1 && partial && row < L && m < 3 * F) {
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

// gesr_select: serve for one given snapshot; grid = (token blocks, layer)
template <int KT>
__global__ void __launch_bounds__(kEvalThreads)
select_kernel(const int16_t* __restrict__ indices, long long N, int k, int E, int P, int r,
              const int8_t* __restrict__ primary, const int8_t* __restrict__ replicas,
              const double* __restrict__ snapshot, float theta, long long token_offset, signed char* __restrict__ serve) {
    extern __shared__ __align__(16) unsigned char ssm[];
    constexpr int KM = KT > 0 ? KT : 16;
    LayerTables T;
    carve_tables(ssm, E, r, T);
    __shared__ unsigned long long feas_s;
    const int layer = blockIdx.y;
    load_tables(E, r, primary + (size_t)layer * E, replicas ? replicas + (size_t)layer * E * r : nullptr, T);
    if (threadIdx.x < 64) T.S[threadIdx.x] = threadIdx.x < P ? snapshot[(size_t)layer * P + threadIdx.x] : 0.0;
    __syncthreads();
    if (threadIdx.x == 0) feas_s = load_guard(T.S, P, theta);
    __syncthreads();
    build_candidates(E, r, T, feas_s);
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

// clears the accumulated outputs and the barrier scratch in one launch
__global__ void eval_zero_kernel(unsigned long long* a, size_t na, unsigned long long* b, size_t nb,
                                 unsigned long long* c, size_t nc, unsigned long long* d, size_t nd,
                                 unsigned long long* s, size_t ns) {
    tacg_pdl_prologue();
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    const size_t i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (size_t i = i0; i < na; i += stride) a[i] = 0ull;
    for (size_t i = i0; i < nb; i += stride) b[i] = 0ull;
    for (size_t i = i0; i < nc; i += stride) c[i] = 0ull;
    for (size_t i = i0; i < nd; i += stride) d[i] = 0ull;
    for (size_t i = i0; i < ns; i += stride) s[i] = 0ull;
}

size_t eval_smem_bytes(int E, int P, int r) {
    return tables_bytes(E, r) + 64 * sizeof(unsigned long long) + sizeof(unsigned) * (size_t)P * 32 +
           (r > 0 ? sizeof(unsigned) * (size_t)(kEvalThreads / 32) * kDeferCap * kDeferWords : 0) +
           sizeof(unsigned) * (size_t)(kEvalThreads / 32) * 8 * 32;
}

template <int KT>
int launch_eval_t(tacg_ctx* ctx, EvalParams& p) {
    const size_t smem = eval_smem_bytes(p.E, p.P, p.r);
    const bool rep = p.replicas != nullptr && p.r > 0;
    const bool out = p.cost != nullptr || p.serve != nullptr;
    void (*kern)(EvalParams);
    if (p.P <= 32) {
        kern = rep ? (out ? eval_kernel<KT, true, unsigned, true> : eval_kernel<KT, true, unsigned, false>)
                   : (out ? eval_kernel<KT, false, unsigned, true> : eval_kernel<KT, false, unsigned, false>);
    } else {
        kern = rep ? (out ? eval_kernel<KT, true, unsigned long long, true> : eval_kernel<KT, true, unsigned long long, false>)
                   : (out ? eval_kernel<KT, false, unsigned long long, true> : eval_kernel<KT, false, unsigned long long, false>);
    }
    int occ = 0;
    // the largest shapes (E = 512, P = 64, r = 8) need a little more than the 48 KB default
    TACG_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    TACG_CUDA_TRY(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, kEvalThreads, smem));
    if (occ < 1) occ = 1;
    const int max_grid = ctx->sm_count * occ;
    // CTAs per layer: spread the grid over the layers; never more CTAs than 512-token slices of a micro-batch
    long long cpl = max(1, max_grid / p.L);
    // (one token per thread and micro-batch is still worth a CTA: with few layers the per-micro-batch
    //  latency chain dominates, measured on config 5: 64 CTAs 2.7 ms, 96-128 CTAs 2.5 ms)
    const long long slices = max(1ll, (min(p.B, p.N) + kEvalThreads - 1) / kEvalThreads);
    if (cpl > slices) cpl = slices;
    p.cpl = (int)cpl;
    if ((min(p.B, p.N) + cpl - 1) / cpl + 32 > 0x7fffffffll) {
        snprintf(ctx->detail, sizeof(ctx->detail), "eval: more than 2^31 tokens per CTA slice");
        return TACG_ERR_SHAPE;
    }
    p.groups = (int)min((long long)p.L, (long long)max_grid / cpl);
    const int grid = p.groups * p.cpl;
    const bool waits = rep && p.cpl > 1 && p.nmb > 1;     // CTAs of a group meet at a barrier per micro-batch
    size_t off = 0;
    if (rep) {
        const size_t o_delta = off; off += tacg_align_up(sizeof(unsigned long long) * (size_t)p.L * (size_t)p.nmb * p.P, 256);
        const size_t o_bar = off;   off += tacg_align_up(sizeof(unsigned) * (size_t)p.L, 256);
        char* base = static_cast<char*>(tacg_scratch(ctx, off));
        if (!base) return TACG_ERR_CUDA;
        p.delta = reinterpret_cast<unsigned long long*>(base + o_delta);
        p.barrier = reinterpret_cast<unsigned*>(base + o_bar);
        p.partial = nullptr;
        const size_t ns = p.cpl > 1 ? off / sizeof(unsigned long long) : 0;
        const int zgrid = (int)max((size_t)1, min((size_t)ctx->sm_count, (ns + 1023) / 1024));
        TACG_CUDA_TRY(ctx, tacg_launch_pdl(eval_zero_kernel, dim3(zgrid), dim3(1024), 0, ctx->stream, p.comm_span,
                                           (size_t)p.L * p.F, p.comm_remote, (size_t)p.L * p.F, p.load, (size_t)p.L * p.P,
                                           p.ntok, (size_t)p.F, reinterpret_cast<unsigned long long*>(base), ns));
        TACG_LAUNCH_CHECK(ctx);
    } else {
        // every (layer, part) row is written by exactly one CTA, so nothing needs clearing
        off = sizeof(unsigned long long) * (size_t)p.L * (size_t)p.cpl * (size_t)(p.P + 3 * p.F);
        char* base = static_cast<char*>(tacg_scratch(ctx, off));
        if (!base) return TACG_ERR_CUDA;
        p.partial = reinterpret_cast<unsigned long long*>(base);
        p.delta = nullptr; p.barrier = nullptr;
    }
    tacg_prof_scope prof(ctx, TACG_PROF_EVAL);
    if (waits) {
        void* args[] = {&p};
        TACG_CUDA_TRY(ctx, cudaLaunchCooperativeKernel((const void*)kern, dim3(grid), dim3(kEvalThreads), args, smem,
                                                       ctx->stream));
        ctx->launches += 1;
    } else {
        TACG_CUDA_TRY(ctx, tacg_launch_pdl(kern, dim3(grid), dim3(kEvalThreads), smem, ctx->stream, p));
        TACG_LAUNCH_CHECK(ctx);
    }
    return TACG_OK;
}

template <int KT>
int launch_select_t(tacg_ctx* ctx, const int16_t* indices, int64_t N, int k, int L, int E, int P,
                    const int8_t* primary, const int8_t* replicas, int r, const double* snapshot, float theta,
                    int64_t token_offset, int8_t* serve) {
    const size_t smem = tables_bytes(E, r);
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
    const unsigned long long* fin_partial = nullptr;   // set when the fairness kernel still has the CTA rows to add
    int fin_cpl = 0;
    if (N > 0) {
        EvalParams p;
        p.indices = indices; p.family = family; p.N = N; p.k = k; p.L = L; p.E = E; p.F = F; p.P = P; p.r = r;
        p.primary = primary; p.replicas = replicas; p.theta = theta; p.rho = rho;
        const bool use_rep = replicas != nullptr && r > 0;
        p.B = (!use_rep || microbatch <= 0 || microbatch > N) ? N : microbatch;
        p.nmb = (N + p.B - 1) / p.B;
        p.token_offset = token_offset;
        p.load_state = load_state;
        p.load = reinterpret_cast<unsigned long long*>(load);
        p.comm_span = reinterpret_cast<unsigned long long*>(comm_span);
        p.comm_remote = reinterpret_cast<unsigned long long*>(comm_remote);
        p.ntok = reinterpret_cast<unsigned long long*>(ntok);
        p.cost = cost_per_token;
        p.serve = reinterpret_cast<signed char*>(serve);
        p.delta = nullptr; p.barrier = nullptr; p.partial = nullptr; p.cpl = 1; p.groups = 1;
        int rc;
        switch (tacg_pick_kt(k, indices)) {
            case 2: rc = launch_eval_t<2>(ctx, p); break;
            case 4: rc = launch_eval_t<4>(ctx, p); break;
            case 6: rc = launch_eval_t<6>(ctx, p); break;
            case 8: rc = launch_eval_t<8>(ctx, p); break;
            default: rc = launch_eval_t<0>(ctx, p); break;
        }
        if (rc != TACG_OK) return rc;
        fin_partial = p.partial;
        fin_cpl = p.cpl;
    }
    TACG_CUDA_TRY(ctx, tacg_launch_pdl(fairness_kernel, dim3(L + 1), dim3(1024), 0, ctx->stream,
                                       reinterpret_cast<unsigned long long*>(load), L, P, fairness, fin_partial, fin_cpl, F,
                                       rho, load_state, reinterpret_cast<unsigned long long*>(comm_span),
                                       reinterpret_cast<unsigned long long*>(comm_remote),
                                       reinterpret_cast<unsigned long long*>(ntok)));
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

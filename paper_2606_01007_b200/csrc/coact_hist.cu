// S1+S2 histogram path (TACG_PATH_HIST): dispatch counts D and pair counts C.
//
// Two kernels, no global atomics:
//   coact_hist_kernel      persistent, one CTA per SM.  A CTA owns a contiguous range of
//                          (layer, token-chunk) items and keeps a PRIVATE strict-upper-triangular
//                          uint32 pair histogram in shared memory (all F families when they fit,
//                          else one family per CTA: the F CTAs of a group walk the same token range at
//                          the same time, each through its family's token list, which three small
//                          kernels build once per call -- the labels are shared by all layers).  Four bank-spread copies of the bins when they fit; for
//                          k = 8 a small token-set table short-cuts repeated expert sets.  The
//                          histogram is written once per (CTA, layer) to a scratch slot.
//   coact_finalize_kernel  grid (E/4, L*F), one warp per output row: sums the slots of the layer (L2
//                          resident), mirrors the triangle into the symmetric C, derives D, adds ntok.
//                          With TACG_ZERO_FIRST it stores (diagonal cleared), otherwise it adds to what
//                          is there (diagonal untouched).
//
// D is not counted with its own atomics.  A token with all k slots valid and distinct puts each of
// its experts into exactly k-1 pair increments, so D[e] = (sum of the pair bins touching e) / (k-1);
// a token with empty slots adds the shortfall to a per-expert correction counter, which makes the
// identity exact for every token (see slow_token()).
//
// Fallback for shapes whose single-family triangle does not fit in shared memory (E > ~330):
// coact_global_kernel, plain global atomics.
#include "tacg_common.cuh"

namespace {

constexpr int kThreads = 1024;           // one CTA per SM
constexpr int kWarps = kThreads / 32;
constexpr int kBatch = 4;                 // tokens per thread whose loads are issued together
constexpr int kRun = 256;                   // items (of kThreads tokens) walked together
constexpr int kRunFam = 256;              // the same in family mode (long runs: the set-up of a run, list bounds and
                                          // 64-bit bases, costs as much as four tokens)

struct HistParams {
    const int16_t* indices;
    const int8_t* family;
    long long N;
    int k, L, E, F;
    int nfg;            // 1: a CTA counts all F families; F: CTA c counts family c % F only
    int Fs;             // families per slot (F or 1)
    int tri;            // E(E-1)/2
    int chunk;          // tokens per work item
    int cps;            // items per layer
    long long T;        // L * cps
    int groups;         // CTAs / nfg; group g owns items [g*T/groups, (g+1)*T/groups)
    unsigned* scratch;  // [(groups+L-1)*nfg][slot_words]
    int slot_words;     // Fs*(tri+E+1) rounded up to 4
    int memo_off;       // byte offset of the token-set table in shared memory, 0 = no table
    int memo_ts;        // table entries per family (power of two)
    const unsigned* perm;   // family mode: [F][N] tokens of each family in increasing order
    const unsigned* boff;   // family mode: [F][cps+1] tokens of family f before item (block of `chunk` tokens) b
};

// R(i) + j is the bin of the pair i < j in a row-major strict upper triangle of an E x E matrix:
// R(i) = i(2E-1-i)/2 - i - 1 = i(2E-3-i)/2 - 1 (the product is always even).
__device__ __forceinline__ int tri_row(int i, int E) { return ((i * (2 * E - 3 - i)) >> 1) - 1; }

__device__ __forceinline__ void cswap(int& a, int& b) {
    const int lo = min(a, b), hi = max(a, b);
    a = lo; b = hi;
}

template <int K>
__device__ __forceinline__ void sort_ids(int (&e)[K]) {
    if constexpr (K == 2) {
        cswap(e[0], e[1]);
    } else if constexpr (K == 4) {
        cswap(e[0], e[1]); cswap(e[2], e[3]); cswap(e[0], e[2]); cswap(e[1], e[3]); cswap(e[1], e[2]);
    } else if constexpr (K == 6) {
        cswap(e[0], e[5]); cswap(e[1], e[3]); cswap(e[2], e[4]);
        cswap(e[1], e[2]); cswap(e[3], e[4]);
        cswap(e[0], e[3]); cswap(e[2], e[5]);
        cswap(e[0], e[1]); cswap(e[2], e[3]); cswap(e[4], e[5]);
        cswap(e[1], e[2]); cswap(e[3], e[4]);
    } else if constexpr (K == 8) {
        cswap(e[0], e[2]); cswap(e[1], e[3]); cswap(e[4], e[6]); cswap(e[5], e[7]);
        cswap(e[0], e[4]); cswap(e[1], e[5]); cswap(e[2], e[6]); cswap(e[3], e[7]);
        cswap(e[0], e[1]); cswap(e[2], e[3]); cswap(e[4], e[5]); cswap(e[6], e[7]);
        cswap(e[2], e[4]); cswap(e[3], e[5]);
        cswap(e[1], e[4]); cswap(e[3], e[6]);
        cswap(e[1], e[2]); cswap(e[3], e[4]); cswap(e[5], e[6]);
    }
}

// Any token: every slot is checked.  For each valid slot a, cnt = number of pair increments the
// slot takes part in; the correction counter receives (k-1) - cnt so that
// (pair bins touching e) + corr[e] = (k-1) * (valid slots holding e)   holds exactly.
template <int KMAX, int CP = 1>
__device__ __forceinline__ void slow_token(const int (&e)[KMAX], int k, int E, unsigned* hist, unsigned* corr) {
    const int km1 = max(k - 1, 1);
    for (int a = 0; a < k; ++a) {
        const int i = e[a];
        if ((unsigned)i >= (unsigned)E) continue;   // empty slot (or id out of range: skipped)
        int cnt = 0;
        for (int b = 0; b < k; ++b) {
            const int j = e[b];
            if (b == a || (unsigned)j >= (unsigned)E || j == i) continue;
            ++cnt;
            if (b > a) {
                TACG_ASSERT(tri_row(min(i, j), E) + max(i, j) >= 0 && tri_row(min(i, j), E) + max(i, j) < E * (E - 1) / 2);
                atomicAdd(&hist[(tri_row(min(i, j), E) + max(i, j)) * CP], 1u);
            }
        }
        if (km1 - cnt) atomicAdd(&corr[i], (unsigned)(km1 - cnt));
    }
}

// Raw 32-bit words of one token row (two ids per word); KT in {2,4,6,8}, base 16-byte aligned.
template <int KT>
__device__ __forceinline__ void load_raw(const int16_t* __restrict__ row, unsigned (&w)[KT / 2]) {
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

// One token (KT ids packed in w) of a family whose triangle starts at hist (corr = its correction counters).
// CP > 1: the bins are interleaved CP-fold (word = bin * CP + copy) and hist already points at this
// lane's copy, so lanes of different copies never share a bank.
// Token-set table (one region per family): a token whose sorted ids are already a key of the table
// costs one 64-bit CAS and one increment instead of k(k-1)/2 bin increments; the entries are expanded
// into the bins (count x every pair) when the CTA leaves the layer.  Exact for any input; it pays
// when expert sets repeat (planted groups, popular sets) and costs one failed CAS otherwise.
struct MemoTable {
    unsigned long long* keys;   // nullptr = disabled; 0 = empty entry (never a key: ids are distinct, k >= 2)
    unsigned* cnt;
    unsigned mask;              // entries - 1
};

template <int KT, int CP = 1>
__device__ __forceinline__ void count_packed(const unsigned (&w)[KT / 2], int E, unsigned* hist, unsigned* corr,
                                             const MemoTable memo = MemoTable{nullptr, nullptr, 0u}) {
    int e[KT], s[KT];
#pragma unroll
    for (int i = 0; i < KT / 2; ++i) {
        e[2 * i] = (int)(short)(w[i] & 0xffffu);
        e[2 * i + 1] = (int)w[i] >> 16;
    }
#pragma unroll
    for (int a = 0; a < KT; ++a) s[a] = e[a];
    sort_ids<KT>(s);
    bool fast = s[0] >= 0 && s[KT - 1] < E;
#pragma unroll
    for (int a = 0; a + 1 < KT; ++a) fast = fast && (s[a] != s[a + 1]);
    if (fast) {
        if (memo.keys) {
            unsigned long long key = 0ull;
#pragma unroll
            for (int a = 0; a < KT; ++a) key |= (unsigned long long)(unsigned)s[a] << (8 * a);
            const unsigned h = (unsigned)((key * 0x9E3779B97F4A7C15ull) >> 40) & memo.mask;
            // plain read first: once a set is in the table a hit costs one load and one increment
            unsigned long long prev = *reinterpret_cast<volatile unsigned long long*>(memo.keys + h);
            if (prev == 0ull) prev = atomicCAS(memo.keys + h, 0ull, key);
            if (prev == 0ull || prev == key) {
                atomicAdd(memo.cnt + h, 1u);
                return;
            }
        }
#pragma unroll
        for (int a = 0; a + 1 < KT; ++a) {
            unsigned* rowp = hist + tri_row(s[a], E) * CP;
#pragma unroll
            for (int b = a + 1; b < KT; ++b) {
                TACG_ASSERT(tri_row(s[a], E) + s[b] >= 0 && tri_row(s[a], E) + s[b] < E * (E - 1) / 2);
                atomicAdd(rowp + s[b] * CP, 1u);
            }
        }
        return;
    }
    slow_token<KT, CP>(e, KT, E, hist, corr);
}

// One token, any k: compile-time KT uses the packed path, KT == 0 reads k ids one by one.
template <int KT, int CP = 1>
__device__ __forceinline__ void count_token(const int16_t* __restrict__ row, int k, int E, unsigned* hist,
                                            unsigned* corr, const MemoTable memo = MemoTable{nullptr, nullptr, 0u}) {
    if constexpr (KT >= 2) {
        unsigned w[KT / 2];
        load_raw<KT>(row, w);
        count_packed<KT, CP>(w, E, hist, corr, memo);
    } else {
        int e[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) e[j] = (j < k) ? (int)__ldg(row + j) : -1;
        slow_token<16, CP>(e, k, E, hist, corr);
    }
}

// Eight ids, two per word, sorted into the eight bytes of a key (smallest id in the lowest byte).
// Lanes: the low halves of the four words are one sequence, the high halves another; both are sorted with the same
// five word-wide compare-exchanges, then merged as a bitonic sequence whose compare-exchanges are again word-wide
// after two byte permutes.  ok = every id is in [0, 256) and no two are equal (else the caller takes the slow path).
__device__ __forceinline__ unsigned long long sort8_key(const unsigned (&w)[4], bool& ok) {
    unsigned a = w[0], b = w[1], c = w[2], d = w[3], t;
    const unsigned orw = (a | b) | (c | d);
    // 4-sorter on the words: (0,1) (2,3) (0,2) (1,3) (1,2)
    t = __vminu2(a, b); b = __vmaxu2(a, b); a = t;
    t = __vminu2(c, d); d = __vmaxu2(c, d); c = t;
    t = __vminu2(a, c); c = __vmaxu2(a, c); a = t;
    t = __vminu2(b, d); d = __vmaxu2(b, d); b = t;
    t = __vminu2(b, c); c = __vmaxu2(b, c); b = t;
    // x = low lane ascending, y = high lane ascending; pair x_i with y_(3-i)
    const unsigned x01 = __byte_perm(a, b, 0x5410), x23 = __byte_perm(c, d, 0x5410);
    const unsigned y32 = __byte_perm(d, c, 0x7632), y10 = __byte_perm(b, a, 0x7632);
    const unsigned l01 = __vminu2(x01, y32), h01 = __vmaxu2(x01, y32);
    const unsigned l23 = __vminu2(x23, y10), h23 = __vmaxu2(x23, y10);
    const unsigned pl = __vminu2(l01, l23), ql = __vmaxu2(l01, l23);     // lower four: (0,2) (1,3)
    const unsigned ph = __vminu2(h01, h23), qh = __vmaxu2(h01, h23);     // upper four
    const unsigned t0 = __byte_perm(pl, ql, 0x5410), t1 = __byte_perm(pl, ql, 0x7632);
    const unsigned u0 = __byte_perm(ph, qh, 0x5410), u1 = __byte_perm(ph, qh, 0x7632);
    const unsigned lo_e = __vminu2(t0, t1), lo_o = __vmaxu2(t0, t1);     // (s0, s2), (s1, s3)
    const unsigned hi_e = __vminu2(u0, u1), hi_o = __vmaxu2(u0, u1);     // (s4, s6), (s5, s7)
    const unsigned k0 = __byte_perm(lo_e, lo_o, 0x6240), k1 = __byte_perm(hi_e, hi_o, 0x6240);
    // neighbours equal <=> a zero byte in key ^ (key >> 8) (the top byte compares s7 with 0: s7 = 0 means all equal)
    const unsigned d0 = k0 ^ __funnelshift_r(k0, k1, 8), d1 = k1 ^ (k1 >> 8);
    const unsigned z = ((d0 - 0x01010101u) & ~d0) | ((d1 - 0x01010101u) & ~d1);
    ok = (orw & 0xff00ff00u) == 0u && (z & 0x80808080u) == 0u;
    return (unsigned long long)k0 | ((unsigned long long)k1 << 32);
}

// smem layout (words): [Fs][tri] pair bins | [Fs][E] corr | [Fs] ntok (layer 0 only) | pad to slot_words
// CP (non-filter mode only): bank-spread copies of the pair bins, one per quarter warp.
template <int KT, bool FILTER, int CP>
__global__ void __launch_bounds__(kThreads, 1) coact_hist_kernel(const HistParams p) {
    tacg_pdl_prologue();
    extern __shared__ __align__(16) unsigned hsm[];
    const int tid = threadIdx.x;
    const int g = FILTER ? blockIdx.x / p.nfg : blockIdx.x;
    const int fg = FILTER ? blockIdx.x % p.nfg : 0;
    const long long lo = group_lo(g, p.T, p.groups), hi = group_lo(g + 1, p.T, p.groups);
    if (lo >= hi) return;
    const int nbins = p.Fs * p.tri;                       // pair bins of a slot
    unsigned* corr = hsm + (size_t)nbins * CP;
    unsigned* sntok = corr + (size_t)p.Fs * p.E;
    const int k = KT > 0 ? KT : p.k;
    uint4* hsm4 = reinterpret_cast<uint4*>(hsm);
    const int tail = p.slot_words - nbins;                 // corr + ntok + padding words
    const int smem4 = (nbins * CP + tail + 3) / 4;
    for (int i = tid; i < smem4; i += kThreads) hsm4[i] = make_uint4(0u, 0u, 0u, 0u);
    __syncthreads();
    unsigned* hist_lane = hsm + (CP > 1 ? ((tid & 31) >> 3) % CP : 0);
    // token-set table: [Fs][memo_ts] keys, then [Fs][memo_ts] counts
    const int mentries = (KT >= 2 && p.memo_off) ? p.Fs * p.memo_ts : 0;
    unsigned long long* mkeys = reinterpret_cast<unsigned long long*>(reinterpret_cast<unsigned char*>(hsm) + p.memo_off);
    unsigned* mcnt = reinterpret_cast<unsigned*>(mkeys + mentries);
    for (int i = tid; i < mentries; i += kThreads) { mkeys[i] = 0ull; mcnt[i] = 0u; }
    auto memo_of = [&](int fl) {
        MemoTable m;
        m.keys = mentries ? mkeys + (size_t)fl * p.memo_ts : nullptr;
        m.cnt = mcnt + (size_t)fl * p.memo_ts;
        m.mask = (unsigned)(p.memo_ts - 1);
        return m;
    };
    // Tokens that miss the token-set table diverge from those that hit it (28 increments against one), so their
    // sorted sets wait in a per-warp queue and are expanded 32 at a time, every lane busy.
    const int lane = tid & 31;
    unsigned long long* qkey = reinterpret_cast<unsigned long long*>(mcnt + mentries + (mentries & 1)) + (tid >> 5) * 64;
    unsigned char* qfam = reinterpret_cast<unsigned char*>(
                              reinterpret_cast<unsigned long long*>(mcnt + mentries + (mentries & 1)) + (kThreads / 32) * 64) +
                          (tid >> 5) * 64;
    int qn = 0;                         // entries waiting in this warp's queue (warp-uniform)
    // pair increments of one sorted set (ids as bytes of `key`), `c` times
    auto expand_key = [&](unsigned long long key, unsigned c, unsigned* hf) {
        if constexpr (KT >= 2) {
            int s[KT];
#pragma unroll
            for (int a = 0; a < KT; ++a) s[a] = (int)((key >> (8 * a)) & 0xffull);
#pragma unroll
            for (int a = 0; a + 1 < KT; ++a) {
                unsigned* rowp = hf + tri_row(s[a], p.E) * CP;
#pragma unroll
                for (int b = a + 1; b < KT; ++b) {
                    TACG_ASSERT(s[a] < s[b] && s[b] < p.E && tri_row(s[a], p.E) + s[b] < p.tri);
                    atomicAdd(rowp + s[b] * CP, c);
                }
            }
        }
    };
    // one token (live = it exists and is not padding) of family slot fl; every lane of the warp calls this together
    auto process = [&](bool live, const unsigned (&w)[KT >= 2 ? KT / 2 : 1], int fl) {
        if constexpr (KT >= 2) {
            if (!mentries) {
                if (live) count_packed<KT, CP>(w, p.E, hist_lane + (size_t)fl * p.tri * CP, corr + fl * p.E);
                return;
            }
            unsigned long long key = 0ull;
            bool miss = false;
            if (live) {
                bool fast;
                if constexpr (KT == 8) {
                    // sorted set as eight bytes without unpacking: the ids stay two per word and every min / max
                    // (VIMNMX.U16x2) orders two pairs at once
                    key = sort8_key(w, fast);
                    fast = fast && (int)(key >> 56) < p.E;
                } else {
                    int s[KT];
#pragma unroll
                    for (int i = 0; i < KT / 2; ++i) {
                        s[2 * i] = (int)(short)(w[i] & 0xffffu);
                        s[2 * i + 1] = (int)w[i] >> 16;
                    }
                    sort_ids<KT>(s);
                    fast = s[0] >= 0 && s[KT - 1] < p.E;
#pragma unroll
                    for (int a = 0; a + 1 < KT; ++a) fast = fast && (s[a] != s[a + 1]);
#pragma unroll
                    for (int a = 0; a < KT; ++a) key |= (unsigned long long)(unsigned)(s[a] & 0xff) << (8 * a);
                }
                if (fast) {
                    const MemoTable memo = memo_of(fl);
                    const unsigned h = (unsigned)((key * 0x9E3779B97F4A7C15ull) >> 40) & memo.mask;
                    // plain read first: once a set is in the table a hit costs one load and one increment
                    unsigned long long prev = *reinterpret_cast<volatile unsigned long long*>(memo.keys + h);
                    if (prev == 0ull) prev = atomicCAS(memo.keys + h, 0ull, key);
                    if (prev == 0ull || prev == key) atomicAdd(memo.cnt + h, 1u);
                    else miss = true;
                } else {
                    int e[KT];
#pragma unroll
                    for (int i = 0; i < KT / 2; ++i) {
                        e[2 * i] = (int)(short)(w[i] & 0xffffu);
                        e[2 * i + 1] = (int)w[i] >> 16;
                    }
                    slow_token<KT, CP>(e, KT, p.E, hist_lane + (size_t)fl * p.tri * CP, corr + fl * p.E);
                }
            }
            const unsigned mm = __ballot_sync(0xffffffffu, miss);
            if (mm) {
                if (miss) {
                    const int pos = qn + __popc(mm & ((1u << lane) - 1u));
                    TACG_ASSERT(pos >= 0 && pos < 64);
                    qkey[pos] = key;
                    qfam[pos] = (unsigned char)fl;
                }
                qn += __popc(mm);
                __syncwarp();
                if (qn >= 32) {
                    qn -= 32;
                    expand_key(qkey[qn + lane], 1u, hist_lane + (size_t)qfam[qn + lane] * p.tri * CP);
                    __syncwarp();
                }
            }
        }
    };
    __syncthreads();


    // Items are walked in runs of up to kRun consecutive items of one layer, so that a thread has
    // kBatch tokens in flight while group boundaries stay at the finer item granularity.
    int layer = (int)(lo / p.cps);
    int ci = (int)(lo - (long long)layer * p.cps);          // item inside the layer
    int l = layer;
    long long item = lo;
    for (;;) {
        if (ci == p.cps) { ci = 0; ++l; }
        if (item == hi) l = -1;
        if (l != layer) {
            const int16_t* lbase = p.indices + (size_t)layer * (size_t)p.N * k;
            if (lane < qn) expand_key(qkey[lane], 1u, hist_lane + (size_t)qfam[lane] * p.tri * CP);   // the rest of the queue
            qn = 0;
            __syncthreads();
            if constexpr (KT >= 2) {
                // expand the token-set table: count x every pair of the key
                for (int i = tid; i < mentries; i += kThreads) {
                    const unsigned c = mcnt[i];
                    if (c) {
                        expand_key(mkeys[i], c, hsm + (size_t)(i / p.memo_ts) * p.tri * CP + (CP > 1 ? (tid & (CP - 1)) : 0));
                        mkeys[i] = 0ull;
                        mcnt[i] = 0u;
                    }
                }
                if (mentries) __syncthreads();
            }
            // flush this (group, layer) visit to its slot, then clear
            unsigned* dst = p.scratch + ((size_t)(g + layer) * p.nfg + fg) * p.slot_words;
            if constexpr (CP == 1) {
                uint4* dst4 = reinterpret_cast<uint4*>(dst);
                for (int i = tid; i < smem4; i += kThreads) {
                    dst4[i] = hsm4[i];
                    hsm4[i] = make_uint4(0u, 0u, 0u, 0u);
                }
            } else {
                static_assert(CP == 1 || CP == 4, "copies are summed with one 16-byte load");
                for (int i = tid; i < nbins; i += kThreads) {
                    const uint4 v = hsm4[i];
                    dst[i] = (v.x + v.y) + (v.z + v.w);
                    hsm4[i] = make_uint4(0u, 0u, 0u, 0u);
                }
                for (int i = tid; i < tail; i += kThreads) {
                    dst[nbins + i] = corr[i];
                    corr[i] = 0u;
                }
            }
            __syncthreads();
            if (l < 0) break;
            layer = l;
        }
        const int run = (int)min((long long)min(FILTER ? kRunFam : kRun, p.cps - ci), hi - item);
        const long long t0 = (long long)ci * p.chunk;
        const long long t1 = min(p.N, t0 + (long long)run * p.chunk);
        ci += run;
        item += run;
        const int16_t* lbase = p.indices + (size_t)l * (size_t)p.N * k;
        if (!FILTER) {
            if constexpr (KT >= 2) {
                // kBatch tokens per thread with all their loads in flight before the first increment
                for (long long tb = t0 + tid; tb - lane < t1; tb += (long long)kThreads * kBatch) {   // warp-uniform trip count
                    int f[kBatch];
                    unsigned w[kBatch][KT / 2];
#pragma unroll
                    for (int u = 0; u < kBatch; ++u) {
                        const long long t = tb + (long long)u * kThreads;
                        f[u] = -1;
                        if (t < t1) {
                            f[u] = p.family[t];
                            load_raw<KT>(lbase + (size_t)t * KT, w[u]);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < kBatch; ++u) {
                        const bool live = (unsigned)f[u] < (unsigned)p.F;    // not a padding token, not past the end
                        if (live && l == 0) atomicAdd(&sntok[f[u]], 1u);
                        process(live, w[u], live ? f[u] : 0);
                    }
                }
            } else {
                for (long long t = t0 + tid; t < t1; t += kThreads) {
                    const int f = p.family[t];
                    if ((unsigned)f >= (unsigned)p.F) continue;     // padding token
                    if (l == 0) atomicAdd(&sntok[f], 1u);
                    count_token<KT, CP>(lbase + (size_t)t * k, k, p.E, hist_lane + (size_t)f * p.tri * CP, corr + f * p.E);
                }
            }
        } else {
            // family mode: the tokens of family fg among [t0, t1) are a contiguous piece of the family's list
            const int b0 = ci - run;
            const unsigned* bo = p.boff + (size_t)fg * (p.cps + 1);
            const unsigned j0 = bo[b0], j1 = bo[b0 + run];
            TACG_ASSERT(b0 >= 0 && b0 + run <= p.cps && j0 <= j1 && (long long)j1 <= p.N);
            const unsigned* __restrict__ list = p.perm + (size_t)fg * (size_t)p.N;
            if (l == 0 && tid == 0) sntok[0] += j1 - j0;
            if constexpr (KT >= 2) {
                // the token ids of a round are read from the list one round ahead: the row gather does not wait for them
                unsigned tok[kBatch];
#pragma unroll
                for (int u = 0; u < kBatch; ++u) {
                    const unsigned j = j0 + tid + u * kThreads;
                    tok[u] = j < j1 ? __ldg(list + j) : 0u;
                }
                for (unsigned jb = j0 + tid; jb - lane < j1; jb += kThreads * kBatch) {     // warp-uniform trip count
                    unsigned w[kBatch][KT / 2];
                    bool live[kBatch];
#pragma unroll
                    for (int u = 0; u < kBatch; ++u) {
                        live[u] = jb + u * kThreads < j1;
                        if (live[u]) load_raw<KT>(lbase + (size_t)tok[u] * KT, w[u]);
                    }
#pragma unroll
                    for (int u = 0; u < kBatch; ++u) {
                        const unsigned jn = jb + (kBatch + u) * kThreads;
                        tok[u] = jn < j1 ? __ldg(list + jn) : 0u;
                    }
#pragma unroll
                    for (int u = 0; u < kBatch; ++u) process(live[u], w[u], 0);
                }
            } else {
                for (unsigned j = j0 + tid; j < j1; j += kThreads)
                    count_token<KT>(lbase + (size_t)__ldg(list + j) * k, k, p.E, hsm, corr);
            }
        }
    }
}

// One warp per output row: grid (ceil(E/4), L*F), 4 rows per CTA (small CTAs: the kernel waits on its loads, and
// measured 4 rows beat 8 and 16).  Each lane sums the slots' bins of its
// (i,j) elements straight from scratch (L2 resident; the four neighbouring rows of a CTA share the
// sectors of the column part), writes the symmetric C row, and the warp reduces the row sum for D.
// ZERO: overwrite instead of accumulate (the diagonal is then cleared with the rest).
template <bool ZERO>
__global__ void __launch_bounds__(128) coact_finalize_kernel(const HistParams p, unsigned* __restrict__ D,
                                                            unsigned* __restrict__ C,
                                                            unsigned long long* __restrict__ ntok) {
    tacg_pdl_prologue();
    const int lf = blockIdx.y;
    const int l = lf / p.F, f = lf % p.F;
    const int E = p.E, tri = p.tri;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i = blockIdx.x * 4 + warp;
    const int fgi = p.nfg > 1 ? f : 0;                   // which CTA of a group holds family f
    const int fs = p.nfg > 1 ? 0 : f;                    // family index inside a slot
    __shared__ int g01[2];                               // first and last group that visited the layer
    if (threadIdx.x == 0) {
        g01[0] = group_of_item((long long)l * p.cps, p.T, p.groups);
        g01[1] = group_of_item((long long)(l + 1) * p.cps - 1, p.T, p.groups);
    }
    __syncthreads();
    const int g0 = g01[0];
    const int ng = g01[1] - g0 + 1;
    const unsigned* slot0 = p.scratch + ((size_t)(g0 + l) * p.nfg + fgi) * p.slot_words;
    const size_t gstride = (size_t)p.nfg * p.slot_words;
    if (l == 0 && blockIdx.x == 0 && warp == 0) {         // slots are read one per lane, then reduced
        unsigned acc = 0;
        for (int g = lane; g < ng; g += 32) acc += slot0[(size_t)g * gstride + (size_t)p.Fs * (tri + E) + fs];
        acc = __reduce_add_sync(0xffffffffu, acc);
        if (lane == 0) ntok[f] = ZERO ? (unsigned long long)acc : ntok[f] + acc;
    }
    if (i >= E) return;
    unsigned* Cf = C + ((size_t)l * p.F + f) * E * E + (size_t)i * E;
    const unsigned* bins = slot0 + (size_t)fs * tri;
    const int ri = tri_row(i, E);
    unsigned rs = 0;
    unsigned corr = 0;
    for (int g = lane; g < ng; g += 32) corr += slot0[(size_t)g * gstride + (size_t)p.Fs * tri + (size_t)fs * E + i];
#pragma unroll 4
    for (int j = lane; j < E; j += 32) {
        unsigned v = 0;
        if (j != i) {
            const unsigned* src = bins + (j > i ? ri + j : tri_row(j, E) + i);
            // eight predicated, independent loads per round: every slot of a typical layer is in flight at once
            unsigned a0 = 0, a1 = 0, a2 = 0, a3 = 0;
            for (int g = 0; g < ng; g += 8) {
                const unsigned* s8 = src + (size_t)g * gstride;
                const int left = ng - g;
                unsigned x[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) x[q] = q < left ? s8[(size_t)q * gstride] : 0u;
                a0 += x[0] + x[4]; a1 += x[1] + x[5]; a2 += x[2] + x[6]; a3 += x[3] + x[7];
            }
            v = (a0 + a1) + (a2 + a3);
        }
        rs += v;
        if (ZERO) Cf[j] = v;
        else if (j != i) Cf[j] += v;
    }
    rs = __reduce_add_sync(0xffffffffu, rs + corr);
    if (lane == 0) {
        const unsigned d = rs / (unsigned)max(p.k - 1, 1);
        unsigned* Df = D + ((size_t)l * p.F + f) * E;
        Df[i] = ZERO ? d : Df[i] + d;
    }
}

// ---- family mode: the tokens of every family as an increasing list, with the list position of every block of
// kThreads tokens (= one work item), built once per call in three small launches.
// (1) boff[f][b] = tokens of family f in block b.  256 threads per block of kThreads tokens, four consecutive tokens each.
constexpr int kPartThreads = kThreads / 4;
constexpr int kPartWarps = kPartThreads / 32;

__device__ __forceinline__ void part_load4(const int8_t* __restrict__ family, long long N, long long t4, int (&f)[4]) {
    if (t4 + 3 < N && ((reinterpret_cast<uintptr_t>(family) + (uintptr_t)t4) & 3u) == 0u) {
        const unsigned v = *reinterpret_cast<const unsigned*>(family + t4);
#pragma unroll
        for (int q = 0; q < 4; ++q) f[q] = (int)(signed char)((v >> (8 * q)) & 0xffu);
    } else {
#pragma unroll
        for (int q = 0; q < 4; ++q) f[q] = t4 + q < N ? (int)family[t4 + q] : -1;
    }
}

__global__ void __launch_bounds__(kPartThreads)
part_count_kernel(const int8_t* __restrict__ family, long long N, int F, int nb, unsigned* __restrict__ boff) {
    tacg_pdl_prologue();
    __shared__ unsigned wc[8][kPartWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int f[4];
    part_load4(family, N, (long long)blockIdx.x * kThreads + (long long)threadIdx.x * 4, f);
    for (int ff = 0; ff < F; ++ff) {
        unsigned c = 0;
#pragma unroll
        for (int q = 0; q < 4; ++q) c += f[q] == ff;
        c = __reduce_add_sync(0xffffffffu, c);
        if (lane == 0) wc[ff][warp] = c;
    }
    __syncthreads();
    if ((int)threadIdx.x < F) {
        unsigned c = 0;
#pragma unroll
        for (int w = 0; w < kPartWarps; ++w) c += wc[threadIdx.x][w];
        boff[(size_t)threadIdx.x * (nb + 1) + blockIdx.x] = c;
    }
}

// (2) in place: boff[f][b] = tokens of family f before block b, boff[f][nb] = all of them; one CTA per family
__global__ void __launch_bounds__(kThreads) part_scan_kernel(int nb, unsigned* __restrict__ boff) {
    tacg_pdl_prologue();
    __shared__ unsigned tsum[kThreads];
    unsigned* row = boff + (size_t)blockIdx.x * (nb + 1);
    const int per = (nb + kThreads - 1) / kThreads;
    const int b0 = min(nb, (int)threadIdx.x * per), b1 = min(nb, b0 + per);
    unsigned s = 0;
    for (int b = b0; b < b1; ++b) s += row[b];
    tsum[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x < 32) {                        // exclusive scan of the 1024 thread sums by one warp
        unsigned carry = 0;
        for (int c = 0; c < kThreads; c += 32) {
            const unsigned v = tsum[c + threadIdx.x];
            unsigned inc = v;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned u = __shfl_up_sync(0xffffffffu, inc, d);
                if ((int)threadIdx.x >= d) inc += u;
            }
            tsum[c + threadIdx.x] = carry + inc - v;
            carry += __shfl_sync(0xffffffffu, inc, 31);
        }
        if (threadIdx.x == 0) row[nb] = carry;
    }
    __syncthreads();
    unsigned run = tsum[threadIdx.x];
    for (int b = b0; b < b1; ++b) {
        const unsigned c = row[b];
        row[b] = run;
        run += c;
    }
}

// (3) perm[f][boff[f][b] + rank of the token among its family's tokens of block b] = token.  The per-thread counts of
// four families travel through one warp scan as 8-bit fields of a word (a warp holds 128 tokens: 128 fits).
__global__ void __launch_bounds__(kPartThreads)
part_scatter_kernel(const int8_t* __restrict__ family, long long N, int F, int nb, const unsigned* __restrict__ boff,
                    unsigned* __restrict__ perm) {
    tacg_pdl_prologue();
    __shared__ unsigned wc[2][kPartWarps];          // warp totals, packed like the scan words
    __shared__ unsigned base_s[8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long t4 = (long long)blockIdx.x * kThreads + (long long)threadIdx.x * 4;
    int f[4];
    part_load4(family, N, t4, f);
    if ((int)threadIdx.x < F) base_s[threadIdx.x] = boff[(size_t)threadIdx.x * (nb + 1) + blockIdx.x];
    unsigned own[2] = {0u, 0u};                     // this thread's tokens per family, packed
#pragma unroll
    for (int q = 0; q < 4; ++q)
        if ((unsigned)f[q] < (unsigned)F) own[f[q] >> 2] += 1u << (8 * (f[q] & 3));
    unsigned inc[2] = {own[0], own[1]};
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned v0 = __shfl_up_sync(0xffffffffu, inc[0], d), v1 = __shfl_up_sync(0xffffffffu, inc[1], d);
        if (lane >= d) { inc[0] += v0; inc[1] += v1; }
    }
    if (lane == 31) { wc[0][warp] = inc[0]; wc[1][warp] = inc[1]; }
    __syncthreads();
    // tokens of each family before this thread in the block: earlier warps (fields up to 128 * 7: sum them unpacked)
    unsigned before[8];
#pragma unroll
    for (int ff = 0; ff < 8; ++ff) {
        unsigned c = ((inc[ff >> 2] - own[ff >> 2]) >> (8 * (ff & 3))) & 0xffu;
        for (int w = 0; w < warp; ++w) c += (wc[ff >> 2][w] >> (8 * (ff & 3))) & 0xffu;
        before[ff] = c;
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int ff = f[q];
        if ((unsigned)ff < (unsigned)F) {
            unsigned r = 0;
#pragma unroll
            for (int x = 0; x < 8; ++x)
                if (x == ff) { r = before[x]; before[x] += 1u; }
            TACG_ASSERT((long long)base_s[ff] + r < N);
            perm[(size_t)ff * (size_t)N + base_s[ff] + r] = (unsigned)(t4 + q);
        }
    }
}

// Fallback: global atomics on D and C (any E <= 512).  The caller zeroes and counts ntok.
__global__ void __launch_bounds__(512)
coact_global_kernel(const int16_t* __restrict__ indices, const int8_t* __restrict__ family, long long N, int k, int L,
                    int E, int F, unsigned* __restrict__ D, unsigned* __restrict__ C) {
    const long long total = (long long)L * N;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long rec = (long long)blockIdx.x * blockDim.x + threadIdx.x; rec < total; rec += stride) {
        const long long l = rec / N, t = rec - l * N;
        const int f = family[t];
        if ((unsigned)f >= (unsigned)F) continue;
        const int16_t* row = indices + (size_t)rec * k;
        unsigned* Dl = D + ((size_t)l * F + f) * E;
        unsigned* Cl = C + ((size_t)l * F + f) * E * E;
        for (int a = 0; a < k; ++a) {
            const int i = row[a];
            if ((unsigned)i >= (unsigned)E) continue;
            atomicAdd(&Dl[i], 1u);
            for (int b = a + 1; b < k; ++b) {
                const int j = row[b];
                if ((unsigned)j >= (unsigned)E || j == i) continue;
                atomicAdd(&Cl[(size_t)i * E + j], 1u);
                atomicAdd(&Cl[(size_t)j * E + i], 1u);
            }
        }
    }
}

template <int KT, bool FILTER, int CP>
int launch_hist(tacg_ctx* ctx, const HistParams& p, size_t smem, int grid) {
    auto kern = coact_hist_kernel<KT, FILTER, CP>;
    TACG_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    TACG_CUDA_TRY(ctx, tacg_launch_pdl(kern, dim3(grid), dim3(kThreads), smem, ctx->stream, p));
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

template <bool FILTER, int CP>
int launch_hist_k(tacg_ctx* ctx, const HistParams& p, size_t smem, int grid) {
    switch (tacg_pick_kt(p.k, p.indices)) {
        case 2: return launch_hist<2, FILTER, CP>(ctx, p, smem, grid);
        case 4: return launch_hist<4, FILTER, CP>(ctx, p, smem, grid);
        case 6: return launch_hist<6, FILTER, CP>(ctx, p, smem, grid);
        case 8: return launch_hist<8, FILTER, CP>(ctx, p, smem, grid);
        default: return launch_hist<0, FILTER, CP>(ctx, p, smem, grid);
    }
}

}  // namespace

int tacg_launch_coact_hist(tacg_ctx* ctx, const int16_t* indices, const int8_t* family, int64_t N, int k, int L,
                           int E, int F, uint32_t* D, uint32_t* C, uint64_t* ntok, bool zero_first) {
    HistParams p;
    p.indices = indices; p.family = family; p.N = N; p.k = k; p.L = L; p.E = E; p.F = F;
    p.tri = E * (E - 1) / 2;
    const size_t limit = (size_t)ctx->smem_optin;
    const size_t all_words = tacg_align_up((size_t)F * (p.tri + E + 1), 4);
    const size_t one_words = tacg_align_up((size_t)(p.tri + E + 1), 4);
    bool filter;
    if (all_words * 4 <= limit) filter = false;
    else if (one_words * 4 <= limit && N < (1ll << 32)) filter = true;
    else {
        // neither layout fits: global atomics
        if (zero_first) {
            TACG_CUDA_TRY(ctx, cudaMemsetAsync(D, 0, sizeof(uint32_t) * (size_t)L * F * E, ctx->stream));
            TACG_CUDA_TRY(ctx, cudaMemsetAsync(C, 0, sizeof(uint32_t) * (size_t)L * F * E * E, ctx->stream));
            TACG_CUDA_TRY(ctx, cudaMemsetAsync(ntok, 0, sizeof(uint64_t) * (size_t)F, ctx->stream));
        }
        int rc = tacg_launch_family_count(ctx, family, N, F, ntok);
        if (rc != TACG_OK) return rc;
        tacg_prof_scope prof(ctx, TACG_PROF_COACT);
        coact_global_kernel<<<ctx->sm_count * 4, 512, 0, ctx->stream>>>(indices, family, (long long)N, k, L, E, F, D, C);
        TACG_LAUNCH_CHECK(ctx);
        return TACG_OK;
    }
    p.nfg = filter ? F : 1;
    p.Fs = filter ? 1 : F;
    p.slot_words = (int)(filter ? one_words : all_words);
    p.chunk = kThreads;
    p.cps = (int)((N + p.chunk - 1) / p.chunk);
    p.T = (long long)L * p.cps;
    // Every (CTA, layer) visit costs one slot (written, then summed by the finalize kernel), so a CTA should
    // own enough items to amortise it: about one item per 12.8 KB of slot (measured on config 5:
    // E = 160, L = 1, N = 1 M tokens: 148 CTAs 107 us, 64 CTAs 57 us, 32 CTAs 63 us).
    const long long min_items = max(2ll, (long long)p.slot_words * 4 / 12800);
    p.groups = (int)max(1ll, min((long long)(ctx->sm_count / p.nfg), max(1ll, p.T / min_items)));
    const size_t slots = (size_t)(p.groups + L - 1) * p.nfg;
    // family mode: the family token lists and their block offsets live behind the slots
    const size_t o_perm = tacg_align_up(slots * p.slot_words * sizeof(unsigned), 256);
    const size_t o_boff = o_perm + (filter ? tacg_align_up(sizeof(unsigned) * (size_t)F * (size_t)N, 256) : 0);
    const size_t total = o_boff + (filter ? sizeof(unsigned) * (size_t)F * ((size_t)p.cps + 1) : 0);
    char* sbase = static_cast<char*>(tacg_scratch(ctx, total));
    if (!sbase) return TACG_ERR_CUDA;
    p.scratch = reinterpret_cast<unsigned*>(sbase);
    p.perm = reinterpret_cast<unsigned*>(sbase + o_perm);
    p.boff = reinterpret_cast<unsigned*>(sbase + o_boff);
    // four bank-spread copies of the pair bins when they fit (non-filter mode)
    const size_t bins_bytes = sizeof(unsigned) * (size_t)p.Fs * p.tri;
    const bool copies = !filter && (size_t)p.slot_words * 4 + 3 * bins_bytes + 16 <= limit;
    size_t smem = (size_t)p.slot_words * 4 + (copies ? 3 * bins_bytes + 16 : 0);
    // token-set table: ids as bytes (E <= 256), packed loaders, 1024 entries per family.  Measured on
    // B200: it pays at k = 8 (28 increments saved per hit: config 3 706 -> 516 us) and loses at k = 6
    // (15 saved, the 64-bit CAS and the key packing cost more: config 2 71 -> 77 us), so k = 8 only.
    p.memo_off = 0;
    p.memo_ts = 1024;
    if (E <= 256 && tacg_pick_kt(k, indices) == 8) {
        const size_t off = tacg_align_up(smem, 16);
        const size_t need = (size_t)p.Fs * p.memo_ts * (sizeof(unsigned long long) + sizeof(unsigned)) + 8 +
                            (size_t)(kThreads / 32) * 64 * (sizeof(unsigned long long) + 1);     // table + the warps' miss queues
        if (off + need <= limit) {
            p.memo_off = (int)off;
            smem = off + need;
        }
    }
    const int grid = p.groups * p.nfg;
    tacg_prof_scope prof(ctx, TACG_PROF_COACT);
    if (filter) {
        unsigned* perm = const_cast<unsigned*>(p.perm);
        unsigned* boff = const_cast<unsigned*>(p.boff);
        TACG_CUDA_TRY(ctx, tacg_launch_pdl(part_count_kernel, dim3(p.cps), dim3(kPartThreads), 0, ctx->stream, family,
                                           (long long)N, F, p.cps, boff));
        TACG_LAUNCH_CHECK(ctx);
        TACG_CUDA_TRY(ctx, tacg_launch_pdl(part_scan_kernel, dim3(F), dim3(kThreads), 0, ctx->stream, p.cps, boff));
        TACG_LAUNCH_CHECK(ctx);
        TACG_CUDA_TRY(ctx, tacg_launch_pdl(part_scatter_kernel, dim3(p.cps), dim3(kPartThreads), 0, ctx->stream, family,
                                           (long long)N, F, p.cps, (const unsigned*)boff, perm));
        TACG_LAUNCH_CHECK(ctx);
    }
    int rc = filter ? launch_hist_k<true, 1>(ctx, p, smem, grid)
                    : (copies ? launch_hist_k<false, 4>(ctx, p, smem, grid) : launch_hist_k<false, 1>(ctx, p, smem, grid));
    if (rc != TACG_OK) return rc;
    unsigned long long* nt = reinterpret_cast<unsigned long long*>(ntok);
    const dim3 fgrid((E + 3) / 4, L * F);
    if (zero_first) TACG_CUDA_TRY(ctx, tacg_launch_pdl(coact_finalize_kernel<true>, fgrid, dim3(128), 0, ctx->stream, p, D, C, nt));
    else TACG_CUDA_TRY(ctx, tacg_launch_pdl(coact_finalize_kernel<false>, fgrid, dim3(128), 0, ctx->stream, p, D, C, nt));
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

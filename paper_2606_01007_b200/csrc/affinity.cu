// S3..S7: preferences (Eq. 2-6), task-modulated graph (Eq. 7-8,
// PAPER.md:97-108), expert->partition affinity (Eq. 10 inner sum) and all-pairs
// swap gains (north_star).  All arithmetic is fp64 on device (DESIGN.md
// "Precision": the z-score divides rounding noise by eps when sigma ~ 0, Q6), results are
// rounded once to fp32 on store.  One launch, a thread-block cluster per layer, four phases:
//   row statistics : per (l,f,i) integer row sums of C and the row maximum of Abar      -> cluster barrier
//   preferences    : per layer, u/c/du/dc/z/s/softmax and max Abar (every CTA its own copy)
//   graph, affinity: W rows and their per-partition segmented sums (aff)                 -> cluster barrier
//   gains          : all-pairs swap gains from aff (fp64 scratch) and W (recomputed in fp64)
// The E x E work is HBM/L2 streaming of C (4*F*E*E bytes per layer); the contraction
// pref.pref^T has inner dimension F <= 8 and W.M is a segmented row sum over a one-hot
// membership matrix, so neither is tensor-core work.
#include <cooperative_groups.h>

#include "tacg_common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int kCluster = 8;        // CTAs per layer (one thread-block cluster)
constexpr int kRowsPerCta = 8;     // one warp per matrix row
constexpr int kRowThreads = kRowsPerCta * 32;

struct AffScratch {
    unsigned long long* rowsum;  // [L,F,E]
    double* rowmax;              // [L,E]
    double* amax;                // [L]
    double* pref64;              // [L,E,F]
    double* aff64;               // [L,E,P]
    double* score64;             // [L,E] GESR score (Eq. 11)
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// Abar[i,j] = (1/F) sum_f C[f,i,j] / max(1,ntok[f])   (readings Q2, Q4).
// inf[f] = 1 / (F * max(1,ntok[f])): one fp64 reciprocal per family instead of a division per entry;
// the result differs from the divided form by a few fp64 ulps, far inside the fp32 tolerance (Q14).
__device__ __forceinline__ double abar_entry(const unsigned* __restrict__ Cl, const double* inf, int F, int E, int i, int j) {
    double s = 0.0;
    for (int f = 0; f < F; ++f) s += (double)__ldg(&Cl[((size_t)f * E + i) * E + j]) * inf[f];
    return s;
}

// W[i,j] of Eq. 8 from Abar, max Abar and the preference rows of i and j (Eq. 7).
// iamax = 1/max Abar (0 when the maximum is 0, Q8).
__device__ __forceinline__ double w_entry(double abar, double iamax, const double* pi, const double* pj, int F, double alpha) {
    const double ah = abar * iamax;
    double at = 0.0;
    for (int f = 0; f < F; ++f) at += pi[f] * pj[f];
    return (1.0 - alpha) * ah + alpha * (at * ah);
}

// relative advantage of family f at one expert: x^f - mean of the other families (Eq. 2-3, Q5)
// inv_others = 1/(F-1) (0 when F = 1): one reciprocal per warp instead of a division per expert
__device__ __forceinline__ double rel_adv(const double* x, int E, int F, int f, int e, double inv_others) {
    double other = 0.0;
    for (int g = 0; g < F; ++g)
        if (g != f) other += x[g * E + e];
    return x[f * E + e] - other * inv_others;
}

// Region A of the fused kernel's shared memory holds first the four F x E work arrays of the preference
// step, later kRowsPerCta W rows and the partition order (E shorts): the larger of the two, in doubles.
__host__ __device__ __forceinline__ size_t region_a_doubles(int E, int F) {
    const size_t pref = (size_t)4 * F * E, graph = (size_t)kRowsPerCta * E + (size_t)(E + 3) / 4;
    return pref > graph ? pref : graph;
}

struct AffArgs {
    const unsigned* C;                 // [L,F,E,E]
    const unsigned* D;                 // [L,F,E]
    const unsigned long long* ntok;    // [F]
    int E, F, P;
    const int8_t* primary;             // [L,E] or NULL
    double alpha, tau, eps;
    AffScratch s;
    float* pref_out;                   // any of the four may be NULL
    float* W_out;
    float* aff_out;
    float* gain_out;
    int need_graph;                    // W, aff or gain wanted (or the GESR step follows)
};

// One thread-block cluster of kCluster CTAs per layer walks S3..S7 in one launch.  Row blocks of
// kRowsPerCta rows (one warp per row) are dealt round-robin to the CTAs of the cluster; the two points
// where a row needs every other row's result (the z-scores of Eq. 4 need all row sums, the gains need all
// affinities) are cluster barriers instead of kernel boundaries.  The preference table is small (E x F),
// so every CTA computes its own copy into shared memory rather than exchanging it.
// Dynamic smem: region A = 4*F*E doubles (u, c, sc, dv of the preference step; afterwards the W rows of
// this CTA's row block and the partition order), region B = E*F doubles (the preference table).
// FT = the family count at compile time (4 and 8: the paper's F = 4 and the ABI maximum), 0 = runtime.
// MINB = CTAs per SM the register budget must allow.  The kernel is bound by the latency of its loads of C: with E >= 256
// (eight rounds per lane) the unrolled loops keep four rounds in flight and want the registers (MINB = 2: 128 of them,
// two CTAs per SM); below that three resident CTAs per SM matter more (MINB = 3: 80 registers).
template <int FT, int MINB>
__global__ void __cluster_dims__(kCluster, 1, 1) __launch_bounds__(kRowThreads, MINB)
affinity_fused_kernel(AffArgs a) {
    tacg_pdl_prologue();
    extern __shared__ double fsm[];
    __shared__ double red[kRowsPerCta];
    __shared__ double amax_s;
    __shared__ int start[65];
    __shared__ double nf_s[8];
    __shared__ short order[512];          // experts sorted by partition (E <= 512)
    cg::cluster_group cluster = cg::this_cluster();
    const int E = a.E, F = FT ? FT : a.F, P = a.P;
    const int l = blockIdx.x / kCluster, rank = blockIdx.x % kCluster;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const AffScratch s = a.s;
    const unsigned* Cl = a.C + (size_t)l * F * E * E;
    const int nblocks = (E + kRowsPerCta - 1) / kRowsPerCta;
    const int8_t* pr = a.primary ? a.primary + (size_t)l * E : nullptr;
    // Up front, off the critical path: the per-family reciprocals (one division each for the CTA, not per
    // thread) and the experts sorted by partition (ascending id inside a partition), one warp per partition:
    // ballots over 32 experts at a time.
    if (threadIdx.x < F) nf_s[threadIdx.x] = 1.0 / ((double)F * (double)max(1ull, a.ntok[threadIdx.x]));
    if (pr && a.need_graph) {
        for (int m = warp; m < P; m += kRowsPerCta) {
            int n = 0;
            for (int e0 = 0; e0 < E; e0 += 32) {
                const int e = e0 + lane;
                n += __popc(__ballot_sync(0xffffffffu, e < E && pr[e] == m));
            }
            if (lane == 0) start[m + 1] = n;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            start[0] = 0;
            for (int m = 0; m < P; ++m) start[m + 1] += start[m];
        }
        __syncthreads();
        for (int m = warp; m < P; m += kRowsPerCta) {
            int pos = start[m];
            for (int e0 = 0; e0 < E; e0 += 32) {
                const int e = e0 + lane;
                const bool mine = e < E && pr[e] == m;
                const unsigned bal = __ballot_sync(0xffffffffu, mine);
                if (mine) order[pos + __popc(bal & ((1u << lane) - 1u))] = (short)e;
                pos += __popc(bal);
            }
        }
    }
    __syncthreads();
    double nf[8];
    for (int f = 0; f < F; ++f) nf[f] = nf_s[f];

    // ---- row sums of C^f and the row maxima of Abar, for this CTA's rows ----
    for (int b = rank; b < nblocks; b += kCluster) {
        const int i = b * kRowsPerCta + warp;
        if (i >= E) continue;
        // one pass over the F rows: integer row sums and the row maximum of Abar together
        double rmax = 0.0;
        unsigned long long acc[8];
#pragma unroll
        for (int f = 0; f < 8; ++f) acc[f] = 0ull;
        // (unrolled: the kernel is bound by the latency of these loads, four rounds of F of them in flight per lane)
#pragma unroll 4
        for (int j = lane; j < E; j += 32) {
            double ab = 0.0;
#pragma unroll
            for (int f = 0; f < 8; ++f) {
                if (f < F) {
                    const unsigned v = __ldg(&Cl[((size_t)f * E + i) * E + j]);
                    acc[f] += v;
                    ab += (double)v * nf[f];
                }
            }
            rmax = fmax(rmax, ab);
        }
        rmax = warp_max(rmax);
#pragma unroll
        for (int f = 0; f < 8; ++f) {
            if (f < F) {
                unsigned long long t = acc[f];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
                if (lane == 0) s.rowsum[((size_t)l * F + f) * E + i] = t;
            }
        }
        if (lane == 0) s.rowmax[(size_t)l * E + i] = rmax;
    }
    cluster.sync();        // release/acquire at cluster scope: the scratch rows written above are visible to the cluster

    // ---- preferences of the whole layer (every CTA its own copy) ----
    double* u = fsm;
    double* c = fsm + (size_t)F * E;
    double* sc = fsm + (size_t)2 * F * E;
    double* dv = fsm + (size_t)3 * F * E;
    double* ptab = fsm + region_a_doubles(E, F);    // [E][F]
    const unsigned* Dl = a.D + (size_t)l * F * E;
    // Warp f owns family f (F <= 8 = warps of the CTA): every sum over experts is a warp reduction.
    // O2: u = D / sum D (Q1), c = rowsum(C)/N_f (Eq. 2 right; counts >= 0 so |.| is the identity, Q3)
    if (warp < F) {
        const int f = warp;
        double part = 0.0;
        for (int e = lane; e < E; e += 32) part += (double)Dl[f * E + e];          // exact: integers < 2^53
        const double itot = 1.0 / fmax(1.0, warp_sum(part));
        const double infam = 1.0 / (double)max(1ull, a.ntok[f]);
        for (int e = lane; e < E; e += 32) {
            u[f * E + e] = (double)Dl[f * E + e] * itot;
            c[f * E + e] = (double)s.rowsum[((size_t)l * F + f) * E + e] * infam;
        }
    }
    __syncthreads();
    // O3, O4: relative advantage (Eq. 2-3) and z-score over experts (Eq. 4).  One warp per (family, quantity):
    // the usage and the co-activation z-scores are independent, so 2F warps work at once; each leaves its
    // z-scores in place of its relative advantages and Eq. 5 adds the two in the softmax below.
    for (int task = warp; task < 2 * F; task += kRowsPerCta) {
        const int f = task % F, pass = task / F;
        const double* x = pass == 0 ? u : c;
        double* dvp = pass == 0 ? sc : dv;
        const double inv_others = F > 1 ? 1.0 / (double)(F - 1) : 0.0;
        double part = 0.0;
        for (int e = lane; e < E; e += 32) {
            const double d = rel_adv(x, E, F, f, e, inv_others);
            dvp[f * E + e] = d;
            part += d;
        }
        const double mu = warp_sum(part) / (double)E;
        double vpart = 0.0;
        for (int e = lane; e < E; e += 32) {
            const double d = dvp[f * E + e] - mu;
            vpart += d * d;
        }
        const double isig = 1.0 / (sqrt(warp_sum(vpart) / (double)E) + a.eps);
        for (int e = lane; e < E; e += 32) dvp[f * E + e] = (dvp[f * E + e] - mu) * isig;
    }
    __syncthreads();
    // O5: temperature softmax over families (Eq. 6), max subtracted
    const double itau = 1.0 / a.tau;
    for (int e = threadIdx.x; e < E; e += kRowThreads) {
        double m = -INFINITY;
        double sv[8];
        for (int f = 0; f < F; ++f) {
            sv[f] = (sc[f * E + e] + dv[f * E + e]) * itau;        // s = z(du) + z(dc), Eq. 5
            m = fmax(m, sv[f]);
        }
        double ex[8];
        double tot = 0.0;
        for (int f = 0; f < F; ++f) {
            ex[f] = exp(sv[f] - m);
            tot += ex[f];
        }
        const double itot = 1.0 / tot;
        for (int f = 0; f < F; ++f) {
            const double p = ex[f] * itot;
            ptab[(size_t)e * F + f] = p;
            if (a.pref_out && rank == 0) a.pref_out[((size_t)l * E + e) * F + f] = (float)p;
        }
    }
    // max Abar over the layer (Q8)
    double mx = 0.0;
    for (int e = threadIdx.x; e < E; e += kRowThreads) mx = fmax(mx, s.rowmax[(size_t)l * E + e]);
    mx = warp_max(mx);
    if (lane == 0) red[warp] = mx;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < kRowsPerCta; ++w) t = fmax(t, red[w]);
        amax_s = t;
    }
    __syncthreads();
    if (!a.need_graph) return;                       // uniform over the cluster

    // ---- W rows (Eq. 8) and their per-partition sums (Eq. 10), for this CTA's rows ----
    const double iamax = amax_s > 0.0 ? 1.0 / amax_s : 0.0;
    double* wrow = fsm;                                                   // region A is free again
    double* wr = wrow + (size_t)warp * E;
    for (int b = rank; b < nblocks; b += kCluster) {
        const int i = b * kRowsPerCta + warp;
        if (i >= E) continue;
        const double* pi = ptab + (size_t)i * F;
#pragma unroll 4
        for (int j = lane; j < E; j += 32) {
            const double w = w_entry(abar_entry(Cl, nf, F, E, i, j), iamax, pi, ptab + (size_t)j * F, F, a.alpha);
            wr[j] = w;
            if (a.W_out) a.W_out[((size_t)l * E + i) * E + j] = (float)w;
        }
        __syncwarp();
        if (pr) {
            // aff[i,m] = sum over the members of partition m, in ascending expert id (Eq. 10 inner sum)
            for (int m = lane; m < P; m += 32) {
                double acc = 0.0;
                for (int q = start[m]; q < start[m + 1]; ++q) acc += wr[order[q]];
                s.aff64[((size_t)l * E + i) * P + m] = acc;
                if (a.aff_out) a.aff_out[((size_t)l * E + i) * P + m] = (float)acc;
            }
        }
        __syncwarp();
    }
    if (!a.gain_out) return;                         // uniform over the cluster
    cluster.sync();        // release/acquire at cluster scope: the scratch rows written above are visible to the cluster

    // ---- all-pairs swap gains from the affinities of both endpoints and W (recomputed in fp64) ----
    const double* affl = s.aff64 + (size_t)l * E * P;
    for (int b = rank; b < nblocks; b += kCluster) {
        const int i = b * kRowsPerCta + warp;
        if (i >= E) continue;
        const double* pi = ptab + (size_t)i * F;
        const int pa = pr[i] & 63;
        // row i of the affinities sits in the warp's registers (lane p holds partitions p and p + 32): two of the four
        // affinity reads of a pair become shuffles
        const double arow0 = lane < P ? affl[(size_t)i * P + lane] : 0.0;
        const double arow1 = lane + 32 < P ? affl[(size_t)i * P + lane + 32] : 0.0;
        const double ai_pa = affl[(size_t)i * P + pa];
#pragma unroll 4
        for (int jb = 0; jb < E; jb += 32) {         // warp-uniform trip count: the shuffles below are by the whole warp
            const int j = min(jb + lane, E - 1);
            const int pb = pr[j] & 63;
            double g = 0.0;
            // (the entry is loaded for every pair, also the 1 in P inside one partition: no branch around the loads)
            const double w = w_entry(abar_entry(Cl, nf, F, E, i, j), iamax, pi, ptab + (size_t)j * F, F, a.alpha);
            const double s0 = __shfl_sync(0xffffffffu, arow0, pb & 31), s1 = __shfl_sync(0xffffffffu, arow1, pb & 31);
            const double ai_pb = pb < 32 ? s0 : s1;
            if (pa != pb) {
                g = ai_pb + affl[(size_t)j * P + pa] - ai_pa - affl[(size_t)j * P + pb] - 2.0 * w;
            }
            if (jb + lane < E) a.gain_out[((size_t)l * E + i) * E + j] = (float)g;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// GESR offline step: Eq. 11 scores and the Eq. 12 replica table.
// One warp per (layer, expert): the F family profiles A^f[e,:] and their mean are walked once and
// every sum is a warp reduction in fp64.  Readings Q29-Q31: cosine with a zero vector
// is 0, "deviation" is the Euclidean norm, ties go to the lower id.
__global__ void __launch_bounds__(kRowThreads)
gesr_score_kernel(const unsigned* __restrict__ C, const unsigned long long* __restrict__ ntok, int E, int F, double lam1,
                  double lam2, AffScratch s, float* __restrict__ terms_out) {
    tacg_pdl_prologue();
    const int l = blockIdx.y;
    const int e = blockIdx.x * kRowsPerCta + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (e >= E) return;
    double inv[8];
    for (int f = 0; f < F; ++f) inv[f] = 1.0 / (double)max(1ull, ntok[f]);
    const unsigned* Cl = C + (size_t)l * F * E * E;
    double cent = 0.0, nm2 = 0.0, dot[8], n2[8], dev2[8];
#pragma unroll
    for (int f = 0; f < 8; ++f) { dot[f] = 0.0; n2[f] = 0.0; dev2[f] = 0.0; }
    const double invF = 1.0 / (double)F;
    for (int j = lane; j < E; j += 32) {
        double a[8], mean = 0.0;
#pragma unroll
        for (int f = 0; f < 8; ++f) {
            a[f] = f < F ? (double)__ldg(&Cl[((size_t)f * E + e) * E + j]) * inv[f] : 0.0;
            mean += a[f];
        }
        mean *= invF;
        cent += mean;
        nm2 += mean * mean;
#pragma unroll
        for (int f = 0; f < 8; ++f) {
            if (f < F) {
                dot[f] += a[f] * mean;
                n2[f] += a[f] * a[f];
                const double d = a[f] - mean;
                dev2[f] += d * d;
            }
        }
    }
    cent = warp_sum(cent);
    nm2 = warp_sum(nm2);
    double cons = 0.0, spec = 0.0;
#pragma unroll
    for (int f = 0; f < 8; ++f) {
        if (f < F) {
            const double dt = warp_sum(dot[f]), nn = warp_sum(n2[f]), dv = warp_sum(dev2[f]);
            if (nn > 0.0 && nm2 > 0.0) cons += dt / (sqrt(nn) * sqrt(nm2));
            spec = fmax(spec, sqrt(dv));
        }
    }
    cons *= invF;
    if (lane == 0) {
        const double score = cent + lam1 * cons - lam2 * spec;
        s.score64[(size_t)l * E + e] = score;
        if (terms_out) {
            float* o = terms_out + ((size_t)l * E + e) * 4;
            o[0] = (float)score; o[1] = (float)cent; o[2] = (float)cons; o[3] = (float)spec;
        }
    }
}

// One CTA per layer: the n_rep experts with the largest score (ties -> lower id), each with the r
// non-primary partitions of largest affinity (ties -> lower id); -1 everywhere else.
__global__ void __launch_bounds__(256)
gesr_pick_kernel(int E, int P, int n_rep, int r, const int8_t* __restrict__ primary, AffScratch s,
                 signed char* __restrict__ replicas) {
    tacg_pdl_prologue();
    __shared__ unsigned char taken[512];
    __shared__ double wbest[8];
    __shared__ int wbest_e[8];
    __shared__ int chosen_s;
    const int l = blockIdx.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    signed char* rep = replicas + (size_t)l * E * r;
    for (int i = threadIdx.x; i < E * r; i += blockDim.x) rep[i] = -1;
    for (int e = threadIdx.x; e < E; e += blockDim.x) taken[e] = 0;
    __syncthreads();
    const double* sc = s.score64 + (size_t)l * E;
    const int rounds = min(n_rep, E);
    for (int it = 0; it < rounds; ++it) {
        double best = 0.0;
        int be = -1;
        for (int e = threadIdx.x; e < E; e += blockDim.x) {
            if (taken[e]) continue;
            const double v = sc[e];
            if (be < 0 || v > best) { best = v; be = e; }            // ascending e: the first maximum is the lowest id
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, best, o);
            const int oe = __shfl_xor_sync(0xffffffffu, be, o);
            if (oe >= 0 && (be < 0 || ov > best || (ov == best && oe < be))) { best = ov; be = oe; }
        }
        if (lane == 0) { wbest[warp] = best; wbest_e[warp] = be; }
        __syncthreads();
        if (threadIdx.x == 0) {
            double b = 0.0;
            int e = -1;
            for (int w = 0; w < 8; ++w) {
                const int oe = wbest_e[w];
                if (oe >= 0 && (e < 0 || wbest[w] > b || (wbest[w] == b && oe < e))) { b = wbest[w]; e = oe; }
            }
            chosen_s = e;
            if (e >= 0) taken[e] = 1;
        }
        __syncthreads();
        const int e = chosen_s;
        if (e >= 0 && warp == 0) {
            // secondaries of expert e: r rounds of arg max over the non-primary partitions (warp 0)
            const int pm = primary[(size_t)l * E + e] & 63;
            const double* af = s.aff64 + ((size_t)l * E + e) * P;
            unsigned long long used = 1ull << pm;
            for (int a = 0; a < r; ++a) {
                double bv = 0.0;
                int bm = -1;
                for (int m = lane; m < P; m += 32) {
                    if ((used >> m) & 1ull) continue;
                    const double v = af[m];
                    if (bm < 0 || v > bv) { bv = v; bm = m; }
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    const double ov = __shfl_xor_sync(0xffffffffu, bv, o);
                    const int om = __shfl_xor_sync(0xffffffffu, bm, o);
                    if (om >= 0 && (bm < 0 || ov > bv || (ov == bv && om < bm))) { bv = ov; bm = om; }
                }
                if (bm < 0) break;                                   // fewer than r other partitions
                used |= 1ull << bm;
                if (lane == 0) rep[(size_t)e * r + a] = (signed char)bm;
            }
        }
        __syncthreads();
    }
}

}  // namespace

int tacg_launch_affinity(tacg_ctx* ctx, const uint32_t* D, const uint32_t* C, const uint64_t* ntok, int L, int E,
                         int F, int P, const int8_t* primary, double alpha, double tau, double eps, float* pref,
                         float* W, float* aff, float* gain, const tacg_gesr_build* gesr) {
    size_t off = 0;
    const size_t o_rowsum = off; off += tacg_align_up(sizeof(unsigned long long) * (size_t)L * F * E, 256);
    const size_t o_rowmax = off; off += tacg_align_up(sizeof(double) * (size_t)L * E, 256);
    const size_t o_amax = off;   off += tacg_align_up(sizeof(double) * (size_t)L, 256);
    const size_t o_pref = off;   off += tacg_align_up(sizeof(double) * (size_t)L * E * F, 256);
    const size_t o_aff = off;    off += tacg_align_up(sizeof(double) * (size_t)L * E * P, 256);
    const size_t o_score = off;  off += tacg_align_up(sizeof(double) * (size_t)L * E, 256);
    char* base = static_cast<char*>(tacg_scratch(ctx, off));
    if (!base) return TACG_ERR_CUDA;
    AffScratch s;
    s.rowsum = reinterpret_cast<unsigned long long*>(base + o_rowsum);
    s.rowmax = reinterpret_cast<double*>(base + o_rowmax);
    s.amax = reinterpret_cast<double*>(base + o_amax);
    s.pref64 = reinterpret_cast<double*>(base + o_pref);
    s.aff64 = reinterpret_cast<double*>(base + o_aff);
    s.score64 = reinterpret_cast<double*>(base + o_score);
    const unsigned long long* nt = reinterpret_cast<const unsigned long long*>(ntok);
    const dim3 rows((E + kRowsPerCta - 1) / kRowsPerCta, L);
    tacg_prof_scope prof(ctx, TACG_PROF_AFFINITY);
    AffArgs a;
    a.C = C; a.D = D; a.ntok = nt; a.E = E; a.F = F; a.P = P; a.primary = primary;
    a.alpha = alpha; a.tau = tau; a.eps = eps; a.s = s;
    a.pref_out = pref; a.W_out = W; a.aff_out = aff; a.gain_out = gain;
    a.need_graph = (W || aff || gain || gesr) ? 1 : 0;
    const size_t smem = sizeof(double) * (region_a_doubles(E, F) + (size_t)E * F);
    auto launch = [&](auto kernel) -> int {
        TACG_CUDA_TRY(ctx, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        TACG_CUDA_TRY(ctx, tacg_launch_pdl(kernel, dim3(L * kCluster), dim3(kRowThreads), smem, ctx->stream, a));
        TACG_LAUNCH_CHECK(ctx);
        return TACG_OK;
    };
    const int rc = F == 4 ? (E >= 256 ? launch(affinity_fused_kernel<4, 2>) : launch(affinity_fused_kernel<4, 3>))
                 : F == 8 ? launch(affinity_fused_kernel<8, 3>) : launch(affinity_fused_kernel<0, 3>);
    if (rc != TACG_OK) return rc;
    if (gesr) {
        TACG_CUDA_TRY(ctx, tacg_launch_pdl(gesr_score_kernel, rows, dim3(kRowThreads), 0, ctx->stream, C, nt, E, F, gesr->lambda1,
                                           gesr->lambda2, s, gesr->terms));
        TACG_LAUNCH_CHECK(ctx);
        TACG_CUDA_TRY(ctx, tacg_launch_pdl(gesr_pick_kernel, dim3(L), dim3(256), 0, ctx->stream, E, P, gesr->n_rep, gesr->r, primary, s,
                                           reinterpret_cast<signed char*>(gesr->replicas)));
        TACG_LAUNCH_CHECK(ctx);
    }
    return TACG_OK;
}

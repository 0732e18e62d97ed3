// Motivation diagnostics of PAPER.md:469 from the counts the hot path already holds:
// the activation Frobenius distance between task families and the Jaccard overlap of their top-k most
// frequently co-activated expert pairs.  One CTA per layer; the top-k pairs of a family are found by an
// exact radix select on the integer counts (four 8-bit passes over the upper triangle of C^f), so the sets
// are the oracle's sets, ties included (smaller (i,j) first: the ordered compaction of the last pass).
#include "tacg_common.cuh"

namespace {

constexpr int kDivThreads = 256;
constexpr int kDivWarps = kDivThreads / 32;

struct DivParams {
    const uint32_t* D;     // [L,F,E]
    const uint32_t* C;     // [L,F,E,E]
    const uint64_t* ntok;  // [F]
    int L, E, F, topk;
    float* frob;           // [L+1,F,F]
    float* jac;            // [L+1,F,F]
    double* sq;            // scratch [L,F,F] squared distances
    double* jl;            // scratch [L,F,F] per-layer Jaccard
};

struct DivShared {
    int hist[256];
    int warp_sum[kDivWarps];
    unsigned prefix, mask;
    int need, take_all, nsel, eq_seen;
    int inter[64];         // [F*F]
    int count[8];          // pairs selected per family
};

__global__ void __launch_bounds__(kDivThreads) family_divergence_kernel(DivParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    DivShared* sh = reinterpret_cast<DivShared*>(smem_raw);
    int* sel = reinterpret_cast<int*>(smem_raw + sizeof(DivShared));   // [F][topk] pair ids i*E+j
    const int E = p.E, F = p.F, k = p.topk, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int l = blockIdx.x;
    const int EE = E * E;

    for (int f = 0; f < F; ++f) {
        const uint32_t* Cf = p.C + ((size_t)l * F + f) * EE;
        if (tid == 0) { sh->prefix = 0u; sh->mask = 0u; sh->need = k; sh->take_all = 0; sh->nsel = 0; sh->eq_seen = 0; }
        // ---- the k-th largest count of the upper triangle, digit by digit ----
        for (int shift = 24; shift >= 0; shift -= 8) {
            for (int d = tid; d < 256; d += kDivThreads) sh->hist[d] = 0;
            __syncthreads();
            const unsigned prefix = sh->prefix, mask = sh->mask;
            for (int idx = tid; idx < EE; idx += kDivThreads) {
                const int i = idx / E, j = idx - i * E;
                if (i >= j) continue;
                const unsigned v = Cf[idx];
                if ((v & mask) == prefix) atomicAdd(&sh->hist[(v >> shift) & 255u], 1);
            }
            __syncthreads();
            if (tid == 0 && !sh->take_all) {
                int cum = 0, d = 255, need = sh->need;
                for (; d >= 0; --d) {
                    if (cum + sh->hist[d] >= need) break;
                    cum += sh->hist[d];
                }
                if (d < 0) sh->take_all = 1;               // fewer than k pairs in all
                else { sh->prefix = prefix | ((unsigned)d << shift); sh->mask = mask | (255u << shift); sh->need = need - cum; }
            }
            __syncthreads();
        }
        // kth = the threshold count; `need` pairs equal to it are taken in (i,j) order; zero counts never
        const unsigned kth = sh->take_all ? 0u : sh->prefix;
        const int need_eq = (sh->take_all || kth == 0u) ? 0 : sh->need;
        __syncthreads();
        for (int base = 0; base < EE; base += kDivThreads) {
            const int idx = base + tid;
            bool gt = false, eq = false;
            if (idx < EE) {
                const int i = idx / E, j = idx - i * E;
                if (i < j) {
                    const unsigned v = Cf[idx];
                    gt = v > kth;
                    eq = need_eq > 0 && v == kth;
                }
            }
            const unsigned bal = __ballot_sync(0xffffffffu, eq);
            if (lane == 0) sh->warp_sum[warp] = __popc(bal);
            __syncthreads();
            int rank = sh->eq_seen + __popc(bal & ((1u << lane) - 1u));
            for (int w = 0; w < warp; ++w) rank += sh->warp_sum[w];
            if (gt || (eq && rank < need_eq)) sel[f * k + atomicAdd(&sh->nsel, 1)] = idx;
            __syncthreads();
            if (tid == 0) {
                int s = 0;
                for (int w = 0; w < kDivWarps; ++w) s += sh->warp_sum[w];
                sh->eq_seen += s;
            }
            __syncthreads();
        }
        if (tid == 0) sh->count[f] = sh->nsel;
        __syncthreads();
    }

    // ---- Jaccard overlap of the sets ----
    for (int t = tid; t < F * F; t += kDivThreads) sh->inter[t] = 0;
    __syncthreads();
    for (int t = tid; t < F * F * k; t += kDivThreads) {
        const int fg = t / k, a = t - fg * k;
        const int f = fg / F, g = fg - f * F;
        if (a >= sh->count[f]) continue;
        const int id = sel[f * k + a];
        bool hit = false;
        for (int b = 0; b < sh->count[g]; ++b) hit |= sel[g * k + b] == id;
        if (hit) atomicAdd(&sh->inter[fg], 1);
    }
    __syncthreads();
    for (int t = tid; t < F * F; t += kDivThreads) {
        const int f = t / F, g = t - f * F;
        const int uni = sh->count[f] + sh->count[g] - sh->inter[t];
        const double jv = uni ? (double)sh->inter[t] / (double)uni : 0.0;
        p.jl[(size_t)l * F * F + t] = jv;
        p.jac[(size_t)l * F * F + t] = (float)jv;
    }
    // ---- activation distance ----
    for (int t = warp; t < F * F; t += kDivWarps) {
        const int f = t / F, g = t - f * F;
        const double nf = fmax(1.0, (double)p.ntok[f]), ng = fmax(1.0, (double)p.ntok[g]);
        const uint32_t* Df = p.D + ((size_t)l * F + f) * E;
        const uint32_t* Dg = p.D + ((size_t)l * F + g) * E;
        double s = 0.0;
        for (int e = lane; e < E; e += 32) {
            const double d = (double)Df[e] / nf - (double)Dg[e] / ng;
            s += d * d;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) {
            p.sq[(size_t)l * F * F + t] = s;
            p.frob[(size_t)l * F * F + t] = (float)sqrt(s);
        }
    }
}

// Row L of both outputs: the distance over the whole [L,E] matrix, the mean overlap over layers.
__global__ void family_divergence_total_kernel(DivParams p) {
    const int t = threadIdx.x, FF = p.F * p.F;
    if (t >= FF) return;
    double s = 0.0, j = 0.0;
    for (int l = 0; l < p.L; ++l) {
        s += p.sq[(size_t)l * FF + t];
        j += p.jl[(size_t)l * FF + t];
    }
    p.frob[(size_t)p.L * FF + t] = (float)sqrt(s);
    p.jac[(size_t)p.L * FF + t] = (float)(j / (double)p.L);
}

}  // namespace

int tacg_launch_divergence(tacg_ctx* ctx, const uint32_t* D, const uint32_t* C, const uint64_t* ntok, int L, int E,
                           int F, int topk, float* frob, float* jaccard) {
    const size_t per = tacg_align_up((size_t)L * F * F * sizeof(double), 256);
    unsigned char* base = static_cast<unsigned char*>(tacg_scratch(ctx, 2 * per));
    if (!base) return TACG_ERR_CUDA;
    DivParams p;
    p.D = D; p.C = C; p.ntok = ntok; p.L = L; p.E = E; p.F = F; p.topk = topk; p.frob = frob; p.jac = jaccard;
    p.sq = reinterpret_cast<double*>(base);
    p.jl = reinterpret_cast<double*>(base + per);
    const size_t smem = sizeof(DivShared) + (size_t)F * topk * sizeof(int);
    family_divergence_kernel<<<L, kDivThreads, smem, ctx->stream>>>(p);
    TACG_LAUNCH_CHECK(ctx);
    family_divergence_total_kernel<<<1, 64, 0, ctx->stream>>>(p);
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

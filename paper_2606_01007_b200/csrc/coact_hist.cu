// S1+S2 histogram path (TACG_PATH_HIST): dispatch counts D and pair counts C by atomic
// increments.  One thread per token; a CTA keeps a private upper-triangular
// uint32 histogram per family in shared memory when it fits and flushes it once with
// global reductions, otherwise it increments global memory directly.
// Also: the family histogram ntok[F] and the TACG_VALIDATE kernels.
#include "tacg_common.cuh"

namespace {

constexpr int kHistThreads = 512;

// index of the unordered pair i < j in a row-major strict upper triangle of an E x E matrix
__device__ __forceinline__ int tri_index(int i, int j, int E) { return i * (2 * E - i - 1) / 2 + (j - i - 1); }

template <int KT, bool SMEM>
__global__ void __launch_bounds__(kHistThreads)
coact_hist_kernel(const int16_t* __restrict__ indices, const int8_t* __restrict__ family, long long N, int k, int L,
                  int E, int F, int ctas_per_layer, unsigned* __restrict__ D, unsigned* __restrict__ C) {
    extern __shared__ unsigned hsm[];   // SMEM: [F][tri] pair bins, then [F][E] dispatch bins
    const int tri = E * (E - 1) / 2;
    const int layer = blockIdx.x / ctas_per_layer;
    const int part = blockIdx.x % ctas_per_layer;
    if (layer >= L) return;
    if (SMEM) {
        for (int i = threadIdx.x; i < F * (tri + E); i += blockDim.x) hsm[i] = 0u;
        __syncthreads();
    }
    unsigned* hD = hsm + (size_t)F * tri;
    const int16_t* base = indices + (size_t)layer * (size_t)N * (size_t)k;
    unsigned* Dl = D + (size_t)layer * F * E;
    unsigned* Cl = C + (size_t)layer * F * E * E;
    // contiguous token slice of this CTA, in units of kHistThreads tokens
    const long long blocks = (N + kHistThreads - 1) / kHistThreads;
    const long long per = (blocks + ctas_per_layer - 1) / ctas_per_layer;
    const long long t_begin = (long long)part * per * kHistThreads;
    long long t_end = t_begin + per * kHistThreads;
    if (t_end > N) t_end = N;
    for (long long t = t_begin + threadIdx.x; t < t_end; t += kHistThreads) {
        const int f = family[t];
        if ((unsigned)f >= (unsigned)F) continue;       // padding token (or out of range: skipped)
        int e[KT > 0 ? KT : 16];
        tacg_load_ids<KT>(base + (size_t)t * k, k, e);
        const int kk = KT > 0 ? KT : k;
#pragma unroll
        for (int a = 0; a < (KT > 0 ? KT : 16); ++a) {
            if (a >= kk) break;
            const int i = e[a];
            if ((unsigned)i >= (unsigned)E) continue;   // empty slot
            if (SMEM) atomicAdd(&hD[f * E + i], 1u);
            else atomicAdd(&Dl[f * E + i], 1u);
#pragma unroll
            for (int b = a + 1; b < (KT > 0 ? KT : 16); ++b) {
                if (b >= kk) break;
                const int j = e[b];
                if ((unsigned)j >= (unsigned)E || j == i) continue;
                if (SMEM) {
                    const int lo = min(i, j), hi = max(i, j);
                    atomicAdd(&hsm[f * tri + tri_index(lo, hi, E)], 1u);
                } else {
                    atomicAdd(&Cl[((size_t)f * E + i) * E + j], 1u);
                    atomicAdd(&Cl[((size_t)f * E + j) * E + i], 1u);
                }
            }
        }
    }
    if (SMEM) {
        __syncthreads();
        for (int idx = threadIdx.x; idx < F * E; idx += blockDim.x) {
            const unsigned v = hD[idx];
            if (v) atomicAdd(&Dl[idx], v);
        }
        for (int idx = threadIdx.x; idx < F * E * E; idx += blockDim.x) {
            const int f = idx / (E * E);
            const int rem = idx - f * E * E;
            const int i = rem / E, j = rem - i * E;
            if (i == j) continue;
            const unsigned v = hsm[f * tri + tri_index(min(i, j), max(i, j), E)];
            if (v) atomicAdd(&Cl[idx], v);
        }
    }
}

__global__ void family_count_kernel(const int8_t* __restrict__ family, long long N, int F,
                                    unsigned long long* __restrict__ ntok) {
    __shared__ unsigned cnt[8];
    if (threadIdx.x < 8) cnt[threadIdx.x] = 0u;
    __syncthreads();
    unsigned mine[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < N; t += stride) {
        const int f = family[t];
#pragma unroll
        for (int g = 0; g < 8; ++g) mine[g] += (f == g) ? 1u : 0u;
    }
#pragma unroll
    for (int g = 0; g < 8; ++g) {
        const unsigned s = __reduce_add_sync(0xffffffffu, mine[g]);
        if ((threadIdx.x & 31) == 0 && s && g < F) atomicAdd(&cnt[g], s);
    }
    __syncthreads();
    if (threadIdx.x < F && cnt[threadIdx.x]) atomicAdd(&ntok[threadIdx.x], (unsigned long long)cnt[threadIdx.x]);
}

// errword[0] = 1 + smallest bad record id, errword[1] = kind of some bad record.
__global__ void validate_trace_kernel(const int16_t* __restrict__ indices, const int8_t* __restrict__ family,
                                      long long N, int k, int L, int E, int F, unsigned long long* err) {
    const long long total = (long long)L * N;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long rec = (long long)blockIdx.x * blockDim.x + threadIdx.x; rec < total; rec += stride) {
        const long long t = rec % N;
        int kind = 0;
        const int f = family[t];
        if (f >= F) kind = 3;                                   // family out of range (negative = padding)
        const int16_t* row = indices + (size_t)rec * k;
        for (int a = 0; a < k && !kind; ++a) {
            const int i = row[a];
            if (i < 0) continue;                                // empty slot
            if (i >= E) { kind = 1; break; }                    // id out of range
            for (int b = a + 1; b < k; ++b)
                if (row[b] == i) { kind = 2; break; }           // duplicate inside a token
        }
        if (kind) {
            atomicMin(err, (unsigned long long)rec + 1ull);
            err[1] = (unsigned long long)kind;
        }
    }
}

__global__ void validate_placement_kernel(int L, int E, int P, int capacity, const int8_t* __restrict__ primary,
                                          const int8_t* __restrict__ replicas, int r, unsigned long long* err) {
    // one CTA per layer
    __shared__ int count[64];
    const int l = blockIdx.x;
    if (threadIdx.x < 64) count[threadIdx.x] = 0;
    __syncthreads();
    for (int e = threadIdx.x; e < E; e += blockDim.x) {
        const int m = primary[(size_t)l * E + e];
        int kind = 0;
        if (m < 0 || m >= P) kind = 1;
        else atomicAdd(&count[m], 1);
        if (!kind && replicas) {
            for (int a = 0; a < r && !kind; ++a) {
                const int c = replicas[((size_t)l * E + e) * r + a];
                if (c < -1 || c >= P) kind = 3;
                else if (c >= 0) {
                    if (c == m) kind = 4;
                    for (int b = a + 1; b < r; ++b)
                        if (replicas[((size_t)l * E + e) * r + b] == c) kind = 5;
                }
            }
        }
        if (kind) {
            atomicMin(err, (unsigned long long)((size_t)l * E + e) + 1ull);
            err[1] = (unsigned long long)kind;
        }
    }
    __syncthreads();
    if (threadIdx.x < P && count[threadIdx.x] > capacity) {
        atomicMin(err, (unsigned long long)((size_t)l * E) + 1ull);
        err[1] = 2ull;                                          // partition over capacity
    }
}

constexpr unsigned long long kNoError = ~0ull;

__global__ void errword_begin(unsigned long long* err) { err[0] = kNoError; err[1] = 0; }
__global__ void errword_end(unsigned long long* err) { if (err[0] == kNoError) err[0] = 0; }

template <int KT>
int launch_hist(tacg_ctx* ctx, const int16_t* indices, const int8_t* family, int64_t N, int k, int L, int E, int F,
                uint32_t* D, uint32_t* C) {
    const size_t tri = (size_t)E * (E - 1) / 2;
    const size_t smem = sizeof(unsigned) * (size_t)F * (tri + E);
    const bool use_smem = smem <= (size_t)ctx->smem_optin - 1024;
    // CTAs: about two waves of one CTA per SM when the histogram is large, more when small
    const int per_sm = use_smem ? (int)max((size_t)1, min((size_t)4, ((size_t)ctx->smem_optin) / (smem + 1024))) : 4;
    int cpl = max(1, (ctx->sm_count * per_sm) / L);
    const long long blocks = (N + kHistThreads - 1) / kHistThreads;
    if ((long long)cpl > blocks) cpl = (int)max(1ll, blocks);
    const int grid = L * cpl;
    tacg_prof_scope prof(ctx, TACG_PROF_COACT);
    if (use_smem) {
        auto kern = coact_hist_kernel<KT, true>;
        TACG_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<grid, kHistThreads, smem, ctx->stream>>>(indices, family, (long long)N, k, L, E, F, cpl, D, C);
    } else {
        coact_hist_kernel<KT, false><<<grid, kHistThreads, 0, ctx->stream>>>(indices, family, (long long)N, k, L, E,
                                                                            F, cpl, D, C);
    }
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

}  // namespace

int tacg_launch_coact_hist(tacg_ctx* ctx, const int16_t* indices, const int8_t* family, int64_t N, int k, int L,
                           int E, int F, uint32_t* D, uint32_t* C) {
    switch (tacg_pick_kt(k, indices)) {
        case 2: return launch_hist<2>(ctx, indices, family, N, k, L, E, F, D, C);
        case 4: return launch_hist<4>(ctx, indices, family, N, k, L, E, F, D, C);
        case 6: return launch_hist<6>(ctx, indices, family, N, k, L, E, F, D, C);
        case 8: return launch_hist<8>(ctx, indices, family, N, k, L, E, F, D, C);
        default: return launch_hist<0>(ctx, indices, family, N, k, L, E, F, D, C);
    }
}

int tacg_launch_family_count(tacg_ctx* ctx, const int8_t* family, int64_t N, int F, uint64_t* ntok) {
    const int threads = 256;
    long long want = (N + threads * 16 - 1) / (threads * 16);
    const int grid = (int)max(1ll, min(want, (long long)ctx->sm_count * 4));
    family_count_kernel<<<grid, threads, 0, ctx->stream>>>(family, (long long)N, F,
                                                           reinterpret_cast<unsigned long long*>(ntok));
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

int tacg_launch_validate_trace(tacg_ctx* ctx, const int16_t* indices, const int8_t* family, int64_t N, int k, int L,
                               int E, int F) {
    errword_begin<<<1, 1, 0, ctx->stream>>>(ctx->errword);
    TACG_LAUNCH_CHECK(ctx);
    const long long total = (long long)L * N;
    const int grid = (int)max(1ll, min((total + 255) / 256, (long long)ctx->sm_count * 8));
    validate_trace_kernel<<<grid, 256, 0, ctx->stream>>>(indices, family, (long long)N, k, L, E, F, ctx->errword);
    TACG_LAUNCH_CHECK(ctx);
    errword_end<<<1, 1, 0, ctx->stream>>>(ctx->errword);
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

int tacg_launch_validate_placement(tacg_ctx* ctx, int L, int E, int P, int capacity, const int8_t* primary,
                                   const int8_t* replicas, int r) {
    errword_begin<<<1, 1, 0, ctx->stream>>>(ctx->errword);
    TACG_LAUNCH_CHECK(ctx);
    validate_placement_kernel<<<L, 128, 0, ctx->stream>>>(L, E, P, capacity, primary, replicas, r, ctx->errword);
    TACG_LAUNCH_CHECK(ctx);
    errword_end<<<1, 1, 0, ctx->stream>>>(ctx->errword);
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

// Small kernels around the traces: the family histogram ntok[F] (used by the evaluator and by the
// global-atomic fallback of the co-activation build) and the TACG_VALIDATE checks.
#include "tacg_common.cuh"

namespace {

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

}  // namespace

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

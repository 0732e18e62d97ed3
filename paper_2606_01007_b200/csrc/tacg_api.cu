// C-ABI entry points of libtacg (include/tacg.h): argument checks on the host, then
// kernel launches on the ctx stream.  No CPU implementation of any step lives here.
#include <new>

#include "tacg_common.cuh"

namespace {

const char* kVersion = "0.1";

int fail(tacg_ctx* ctx, int code, const char* what) {
    if (ctx) snprintf(ctx->detail, sizeof(ctx->detail), "%s", what);
    return code;
}

// Reads back the device error word written by the validation kernels (one sync).
int read_errword(tacg_ctx* ctx, int code_if_set, const char* what) {
    unsigned long long h[2] = {0, 0};
    TACG_CUDA_TRY(ctx, cudaMemcpyAsync(h, ctx->errword, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
    TACG_CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    if (h[0] != 0) {
        snprintf(ctx->detail, sizeof(ctx->detail), "%s: first bad record %llu (kind %llu)", what, h[0] - 1, h[1]);
        return code_if_set;
    }
    return TACG_OK;
}

bool shape_ok_common(int64_t N, int k, int L, int E) {
    return N >= 0 && k >= 1 && k <= 16 && L >= 1 && E >= 1 && E <= 512;
}

}  // namespace

void* tacg_scratch(tacg_ctx* ctx, size_t bytes) {
    if (bytes <= ctx->scratch_bytes) return ctx->scratch;
    if (ctx->scratch) {
        cudaStreamSynchronize(ctx->stream);
        cudaFree(ctx->scratch);
        ctx->scratch = nullptr;
        ctx->scratch_bytes = 0;
    }
    size_t want = tacg_align_up(bytes, (size_t)1 << 20);
    cudaError_t e = cudaMalloc(&ctx->scratch, want);
    if (e != cudaSuccess) {
        snprintf(ctx->detail, sizeof(ctx->detail), "cudaMalloc(%zu) for scratch: %s", want, cudaGetErrorString(e));
        ctx->scratch = nullptr;
        return nullptr;
    }
    ctx->scratch_bytes = want;
    return ctx->scratch;
}

extern "C" {

const char* tacg_version(void) { return kVersion; }

const char* tacg_strerror(int code) {
    switch (code) {
        case TACG_OK: return "ok";
        case TACG_ERR_NULL: return "a required pointer is NULL";
        case TACG_ERR_SHAPE: return "a size argument is outside the supported limits";
        case TACG_ERR_BAD_INDEX: return "bad expert id, duplicate expert in a token, or bad family (TACG_VALIDATE)";
        case TACG_ERR_PLACEMENT: return "bad primary map or replica table (TACG_VALIDATE)";
        case TACG_ERR_CUDA: return "a CUDA runtime call failed (see tacg_last_detail)";
        case TACG_ERR_ARCH: return "the device is not compute capability 10.x (sm_100)";
        default: return "unknown tacg status";
    }
}

int tacg_create(tacg_ctx** out, int device, void* cuda_stream) {
    if (!out) return TACG_ERR_NULL;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || count <= 0) {
        cudaGetLastError();
        return TACG_ERR_ARCH;   // no CUDA device: there is no CPU fallback
    }
    if (device < 0 || device >= count) return TACG_ERR_SHAPE;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return TACG_ERR_CUDA;
    if (prop.major != 10) return TACG_ERR_ARCH;
    if (cudaSetDevice(device) != cudaSuccess) return TACG_ERR_CUDA;
    tacg_ctx* ctx = new (std::nothrow) tacg_ctx();
    if (!ctx) return TACG_ERR_CUDA;
    ctx->device = device;
    ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    ctx->sm_count = prop.multiProcessorCount;
    ctx->smem_optin = (int)prop.sharedMemPerBlockOptin;
    ctx->scratch = nullptr;
    ctx->scratch_bytes = 0;
    ctx->detail[0] = 0;
    ctx->last_path = 0;
    ctx->launches = 0;
    ctx->profiling = false;
    if (cudaMalloc(&ctx->errword, 2 * sizeof(unsigned long long)) != cudaSuccess) {
        delete ctx;
        return TACG_ERR_CUDA;
    }
    *out = ctx;
    return TACG_OK;
}

int tacg_destroy(tacg_ctx* ctx) {
    if (!ctx) return TACG_ERR_NULL;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    for (int sl = 0; sl < TACG_PROF_SLOTS; ++sl)
        for (auto& pr : ctx->prof[sl]) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
    if (ctx->scratch) cudaFree(ctx->scratch);
    if (ctx->errword) cudaFree(ctx->errword);
    delete ctx;
    return TACG_OK;
}

int tacg_last_detail(tacg_ctx* ctx, char* buf, size_t n) {
    if (!ctx || !buf) return TACG_ERR_NULL;
    if (n == 0) return TACG_OK;
    strncpy(buf, ctx->detail, n - 1);
    buf[n - 1] = 0;
    return TACG_OK;
}

int tacg_profile_enable(tacg_ctx* ctx, int on) {
    if (!ctx) return TACG_ERR_NULL;
    ctx->profiling = on != 0;
    return TACG_OK;
}

int tacg_profile_read(tacg_ctx* ctx, int slot, double* total_ms, int64_t* launches) {
    if (!ctx || !total_ms || !launches) return TACG_ERR_NULL;
    if (slot < 0 || slot >= TACG_PROF_SLOTS) return TACG_ERR_SHAPE;
    double tot = 0.0;
    int64_t n = 0;
    for (auto& pr : ctx->prof[slot]) {
        float ms = 0.f;
        if (cudaEventSynchronize(pr.second) == cudaSuccess && cudaEventElapsedTime(&ms, pr.first, pr.second) == cudaSuccess) {
            tot += ms;
            n += 1;
        }
        cudaEventDestroy(pr.first);
        cudaEventDestroy(pr.second);
    }
    ctx->prof[slot].clear();
    *total_ms = tot;
    *launches = n;
    return TACG_OK;
}

int tacg_last_path(tacg_ctx* ctx) { return ctx ? ctx->last_path : TACG_ERR_NULL; }

int64_t tacg_launch_count(tacg_ctx* ctx) { return ctx ? ctx->launches : (int64_t)TACG_ERR_NULL; }

int tacg_coact_accumulate(tacg_ctx* ctx, const int16_t* indices, const int8_t* family, int64_t N, int k, int L,
                          int E, int F, uint32_t* D, uint32_t* C, uint64_t* ntok, uint32_t flags) {
    if (!ctx) return TACG_ERR_NULL;
    if (!shape_ok_common(N, k, L, E) || F < 1 || F > 8) return fail(ctx, TACG_ERR_SHAPE, "coact: k/L/E/F/N out of range");
    if (!D || !C || !ntok || (N > 0 && (!indices || !family))) return fail(ctx, TACG_ERR_NULL, "coact: NULL pointer");
    const uint32_t path = flags & TACG_PATH_MASK;
    if (path == TACG_PATH_MASK) return fail(ctx, TACG_ERR_SHAPE, "coact: both TACG_PATH_HIST and TACG_PATH_MMA set");
    const bool mma_ok = tacg_coact_mma_supported(k, E, F) && (reinterpret_cast<uintptr_t>(indices) % 16) == 0;
    if (path == TACG_PATH_MMA && !mma_ok)
        return fail(ctx, TACG_ERR_SHAPE, "coact: TACG_PATH_MMA needs k in {2,4,6,8}, E <= 256 and 16-byte aligned indices");
    TACG_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    if ((flags & TACG_VALIDATE) && N > 0) {
        int rc = tacg_launch_validate_trace(ctx, indices, family, N, k, L, E, F);
        if (rc != TACG_OK) return rc;
        rc = read_errword(ctx, TACG_ERR_BAD_INDEX, "coact validate (record = layer*N + token)");
        if (rc != TACG_OK) return rc;
    }
    // Path choice: measured on B200 the histogram kernel is faster than the
    // tensor path at every supported shape, so AUTO takes the histogram; TACG_PATH_MMA forces tcgen05.
    const bool use_mma = N > 0 && path == TACG_PATH_MMA;
    const bool zero_first = (flags & TACG_ZERO_FIRST) != 0;
    if (zero_first && N == 0) {
        TACG_CUDA_TRY(ctx, cudaMemsetAsync(D, 0, sizeof(uint32_t) * (size_t)L * F * E, ctx->stream));
        TACG_CUDA_TRY(ctx, cudaMemsetAsync(C, 0, sizeof(uint32_t) * (size_t)L * F * E * E, ctx->stream));
        TACG_CUDA_TRY(ctx, cudaMemsetAsync(ntok, 0, sizeof(uint64_t) * (size_t)F, ctx->stream));
    }
    if (N == 0) return TACG_OK;
    if (use_mma) {
        ctx->last_path = TACG_PATH_MMA;
        return tacg_launch_coact_mma(ctx, indices, family, N, k, L, E, F, D, C, ntok, zero_first);
    }
    ctx->last_path = TACG_PATH_HIST;
    return tacg_launch_coact_hist(ctx, indices, family, N, k, L, E, F, D, C, ntok, zero_first);
}

int tacg_affinity_swapgain(tacg_ctx* ctx, const uint32_t* D, const uint32_t* C, const uint64_t* ntok, int L, int E,
                           int F, int P, int capacity, const int8_t* primary, float alpha, float tau, float eps,
                           float* pref, float* W, float* aff, float* gain) {
    if (!ctx) return TACG_ERR_NULL;
    if (L < 1 || E < 1 || E > 512 || F < 1 || F > 8) return fail(ctx, TACG_ERR_SHAPE, "affinity: L/E/F out of range");
    if (!D || !C || !ntok) return fail(ctx, TACG_ERR_NULL, "affinity: NULL D/C/ntok");
    if ((aff || gain) && !primary) return fail(ctx, TACG_ERR_NULL, "affinity: aff/gain requested without primary");
    if (primary) {
        if (P < 1 || P > 64 || capacity < 1 || (int64_t)E > (int64_t)P * capacity)
            return fail(ctx, TACG_ERR_SHAPE, "affinity: P out of range or E > P*capacity");
    }
    if (!(tau > 0.0f) || !(eps >= 0.0f)) return fail(ctx, TACG_ERR_SHAPE, "affinity: tau must be > 0 and eps >= 0");
    TACG_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    return tacg_launch_affinity(ctx, D, C, ntok, L, E, F, primary ? P : 1, primary, (double)alpha, (double)tau,
                                (double)eps, pref, W, aff, gain);
}

int gesr_build_replicas(tacg_ctx* ctx, const uint32_t* D, const uint32_t* C, const uint64_t* ntok, int L, int E, int F,
                        int P, int capacity, const int8_t* primary, float alpha, float tau, float eps, float lambda1,
                        float lambda2, int n_rep, int r, int8_t* replicas, float* terms) {
    if (!ctx) return TACG_ERR_NULL;
    if (L < 1 || E < 1 || E > 512 || F < 1 || F > 8) return fail(ctx, TACG_ERR_SHAPE, "gesr_build: L/E/F out of range");
    if (!D || !C || !ntok || !primary || !replicas) return fail(ctx, TACG_ERR_NULL, "gesr_build: NULL pointer");
    if (P < 1 || P > 64 || capacity < 1 || (int64_t)E > (int64_t)P * capacity)
        return fail(ctx, TACG_ERR_SHAPE, "gesr_build: P out of range or E > P*capacity");
    if (n_rep < 0 || r < 1 || r > 8) return fail(ctx, TACG_ERR_SHAPE, "gesr_build: n_rep < 0 or r outside [1,8]");
    if (!(tau > 0.0f) || !(eps >= 0.0f)) return fail(ctx, TACG_ERR_SHAPE, "gesr_build: tau must be > 0 and eps >= 0");
    TACG_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    tacg_gesr_build g;
    g.lambda1 = (double)lambda1; g.lambda2 = (double)lambda2; g.n_rep = n_rep; g.r = r;
    g.replicas = replicas; g.terms = terms;
    return tacg_launch_affinity(ctx, D, C, ntok, L, E, F, P, primary, (double)alpha, (double)tau, (double)eps, nullptr,
                                nullptr, nullptr, nullptr, &g);
}

int tacg_spectral_place(tacg_ctx* ctx, const float* W, int L, int E, int P, int capacity, double jitter,
                        int kmeans_iters, const int8_t* labels_in, int8_t* primary, int8_t* labels0, double* embed) {
    if (!ctx) return TACG_ERR_NULL;
    if (L < 1 || E < 1 || E > 512) return fail(ctx, TACG_ERR_SHAPE, "spectral_place: L/E out of range");
    if (!W || !primary) return fail(ctx, TACG_ERR_NULL, "spectral_place: NULL pointer");
    if (P < 1 || P > 64 || P > E || capacity < 1 || (int64_t)E > (int64_t)P * capacity)
        return fail(ctx, TACG_ERR_SHAPE, "spectral_place: P outside [1, min(64,E)] or E > P*capacity");
    // jitter = 0 would give an expert that never co-activates degree 0 and a NaN in D^-1/2 A D^-1/2
    if (!(jitter > 0.0) || kmeans_iters < 1) return fail(ctx, TACG_ERR_SHAPE, "spectral_place: jitter <= 0 or kmeans_iters < 1");
    TACG_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    return tacg_launch_spectral(ctx, W, L, E, P, capacity, jitter, kmeans_iters, labels_in, primary, labels0, embed);
}

int tacg_family_divergence(tacg_ctx* ctx, const uint32_t* D, const uint32_t* C, const uint64_t* ntok, int L, int E,
                           int F, int topk, float* frob, float* jaccard) {
    if (!ctx) return TACG_ERR_NULL;
    if (L < 1 || E < 1 || E > 512 || F < 1 || F > 8 || topk < 1 || topk > 256)
        return fail(ctx, TACG_ERR_SHAPE, "family_divergence: L/E/F/topk out of range");
    if (!D || !C || !ntok || !frob || !jaccard) return fail(ctx, TACG_ERR_NULL, "family_divergence: NULL pointer");
    TACG_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    return tacg_launch_divergence(ctx, D, C, ntok, L, E, F, topk, frob, jaccard);
}

int gesr_select(tacg_ctx* ctx, const int16_t* indices, int64_t N, int k, int L, int E, int P, const int8_t* primary,
                const int8_t* replicas, int r, const double* load_snapshot, float theta, int64_t token_offset,
                int8_t* serve, uint32_t flags) {
    if (!ctx) return TACG_ERR_NULL;
    if (!shape_ok_common(N, k, L, E) || P < 1 || P > 64 || r < 0 || r > 8 || token_offset < 0)
        return fail(ctx, TACG_ERR_SHAPE, "gesr_select: size out of range");
    if (!primary || !load_snapshot || (N > 0 && (!indices || !serve)))
        return fail(ctx, TACG_ERR_NULL, "gesr_select: NULL pointer");
    if (!replicas) r = 0;
    TACG_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    if (flags & TACG_VALIDATE) {
        int rc = tacg_launch_validate_placement(ctx, L, E, P, E /* capacity not known here */, primary, replicas, r);
        if (rc != TACG_OK) return rc;
        rc = read_errword(ctx, TACG_ERR_PLACEMENT, "gesr_select validate (record = layer*E + expert)");
        if (rc != TACG_OK) return rc;
    }
    if (N == 0) return TACG_OK;
    return tacg_launch_select(ctx, indices, N, k, L, E, P, primary, r ? replicas : nullptr, r, load_snapshot, theta,
                              token_offset, serve);
}

int tacg_eval_placement(tacg_ctx* ctx, const int16_t* indices, const int8_t* family, int64_t N, int k, int L, int E,
                        int F, int P, const int8_t* primary, const int8_t* replicas, int r, float theta, double rho,
                        int64_t microbatch, int64_t token_offset, double* load_state, uint64_t* load,
                        uint64_t* comm_span, uint64_t* comm_remote, uint64_t* ntok, float* fairness,
                        uint8_t* cost_per_token, int8_t* serve, uint32_t flags) {
    if (!ctx) return TACG_ERR_NULL;
    if (!shape_ok_common(N, k, L, E) || F < 1 || F > 8 || P < 1 || P > 64 || r < 0 || r > 8 || token_offset < 0)
        return fail(ctx, TACG_ERR_SHAPE, "eval: size out of range");
    if (!primary || !load || !comm_span || !comm_remote || !ntok || !fairness || (N > 0 && (!indices || !family)))
        return fail(ctx, TACG_ERR_NULL, "eval: NULL pointer");
    if (!replicas) r = 0;
    TACG_CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    if (flags & TACG_VALIDATE) {
        int rc = tacg_launch_validate_placement(ctx, L, E, P, E, primary, replicas, r);
        if (rc != TACG_OK) return rc;
        rc = read_errword(ctx, TACG_ERR_PLACEMENT, "eval validate (record = layer*E + expert)");
        if (rc != TACG_OK) return rc;
    }
    return tacg_launch_eval(ctx, indices, family, N, k, L, E, F, P, primary, r ? replicas : nullptr, r, theta, rho,
                            microbatch, token_offset, load_state, load, comm_span, comm_remote, ntok, fairness,
                            cost_per_token, serve);
}

}  // extern "C"

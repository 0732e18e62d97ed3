// Internal declarations shared by the translation units of libtacg (CUDA path only;
// nothing here is shared with oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include <utility>
#include <vector>

#include "tacg.h"

struct tacg_ctx {
    int device;
    cudaStream_t stream;
    int sm_count;
    int smem_optin;        // max dynamic shared memory per block (opt-in), bytes
    void* scratch;         // grows on demand, reused across calls
    size_t scratch_bytes;
    unsigned long long* errword;  // device: [0] = first bad record + 1 (0 = none), [1] = kind
    char detail[256];
    int last_path;
    int64_t launches;
    bool profiling;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof[TACG_PROF_SLOTS];
};

// Event brackets around the library's own kernels (tacg_profile_enable); no-ops when off.
struct tacg_prof_scope {
    tacg_ctx* ctx;
    int slot;
    cudaEvent_t e0, e1;
    tacg_prof_scope(tacg_ctx* c, int s) : ctx(c), slot(s), e0(nullptr), e1(nullptr) {
        if (ctx->profiling && cudaEventCreate(&e0) == cudaSuccess && cudaEventCreate(&e1) == cudaSuccess)
            cudaEventRecord(e0, ctx->stream);
        else
            e0 = e1 = nullptr;
    }
    ~tacg_prof_scope() {
        if (e1) {
            cudaEventRecord(e1, ctx->stream);
            ctx->prof[slot].emplace_back(e0, e1);
        }
    }
};

#define TACG_CUDA_TRY(ctx, expr)                                                        \
    do {                                                                                \
        cudaError_t _e = (expr);                                                        \
        if (_e != cudaSuccess) {                                                        \
            snprintf((ctx)->detail, sizeof((ctx)->detail), "%s: %s (%s:%d)", #expr,     \
                     cudaGetErrorString(_e), __FILE__, __LINE__);                       \
            return TACG_ERR_CUDA;                                                       \
        }                                                                               \
    } while (0)

#define TACG_LAUNCH_CHECK(ctx)                  \
    do {                                        \
        (ctx)->launches += 1;                   \
        TACG_CUDA_TRY(ctx, cudaGetLastError()); \
    } while (0)

// Returns a device scratch pointer of at least `bytes` (256-byte aligned), or nullptr
// after recording the CUDA error text in ctx->detail.
void* tacg_scratch(tacg_ctx* ctx, size_t bytes);

static inline size_t tacg_align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ---- launchers (each returns a tacg_status) ----
int tacg_launch_family_count(tacg_ctx* ctx, const int8_t* family, int64_t N, int F, uint64_t* ntok);
int tacg_launch_validate_trace(tacg_ctx* ctx, const int16_t* indices, const int8_t* family, int64_t N,
                               int k, int L, int E, int F);
int tacg_launch_validate_placement(tacg_ctx* ctx, int L, int E, int P, int capacity,
                                   const int8_t* primary, const int8_t* replicas, int r);
// Counts D, C and ntok (all three); zero_first = overwrite instead of accumulate.
int tacg_launch_coact_hist(tacg_ctx* ctx, const int16_t* indices, const int8_t* family, int64_t N, int k,
                           int L, int E, int F, uint32_t* D, uint32_t* C, uint64_t* ntok, bool zero_first);
bool tacg_coact_mma_supported(int k, int E, int F);
int tacg_launch_coact_mma(tacg_ctx* ctx, const int16_t* indices, const int8_t* family, int64_t N, int k,
                          int L, int E, int F, uint32_t* D, uint32_t* C, uint64_t* ntok, bool zero_first);
// Optional GESR offline step run after the affinity kernels (gesr_build_replicas).
struct tacg_gesr_build {
    double lambda1, lambda2;
    int n_rep, r;
    int8_t* replicas;   // dev [L,E,r] out
    float* terms;       // dev [L,E,4] out or NULL: (score, Cent, Cons, Spec)
};
int tacg_launch_affinity(tacg_ctx* ctx, const uint32_t* D, const uint32_t* C, const uint64_t* ntok, int L,
                         int E, int F, int P, const int8_t* primary, double alpha, double tau, double eps,
                         float* pref, float* W, float* aff, float* gain, const tacg_gesr_build* gesr = nullptr);
// Spectral-then-repair primary placement (tacg_spectral_place).
int tacg_launch_spectral(tacg_ctx* ctx, const float* W, int L, int E, int P, int capacity, double jitter, int iters,
                         const int8_t* labels_in, int8_t* primary, int8_t* labels0, double* embed);
// Family-divergence diagnostics (tacg_family_divergence).
int tacg_launch_divergence(tacg_ctx* ctx, const uint32_t* D, const uint32_t* C, const uint64_t* ntok, int L, int E,
                           int F, int topk, float* frob, float* jaccard);
int tacg_launch_select(tacg_ctx* ctx, const int16_t* indices, int64_t N, int k, int L, int E, int P,
                       const int8_t* primary, const int8_t* replicas, int r, const double* snapshot,
                       float theta, int64_t token_offset, int8_t* serve);
int tacg_launch_eval(tacg_ctx* ctx, const int16_t* indices, const int8_t* family, int64_t N, int k, int L,
                     int E, int F, int P, const int8_t* primary, const int8_t* replicas, int r, float theta,
                     double rho, int64_t microbatch, int64_t token_offset, double* load_state,
                     uint64_t* load, uint64_t* comm_span, uint64_t* comm_remote, uint64_t* ntok, float* fairness,
                     uint8_t* cost_per_token, int8_t* serve);

// ---- device helpers ----
#ifdef __CUDACC__
// Bounds assertions of the kernels' shared-memory and scratch indices.  compute-sanitizer is closed on the B200 pool
// this library is developed on, so the checks it would make are written into the kernels and switched on with
// TACG_CHECKED=1 python -m paper_2606_01007_b200.build --force (device assert: a violation aborts the launch and the
// next CUDA call returns an error, which every test then reports); they compile to nothing otherwise.
#ifdef TACG_CHECKED
#include <cassert>
#define TACG_ASSERT(x) assert(x)
#else
#define TACG_ASSERT(x) ((void)0)
#endif
// Programmatic dependent launch: the kernels of one step are launched with tacg_launch_pdl and begin with
// tacg_pdl_prologue(), which blocks until the PREVIOUS kernel of the stream has completed and its memory is
// visible.  Everything after the prologue is ordered exactly as with plain stream serialisation; what is saved
// is the drain-and-dispatch gap between small dependent kernels (the dependent grid is set up while its
// predecessor finishes).  No kernel triggers its dependents early: measured, an early trigger packs the next
// kernel's CTAs onto the first SMs that free up and costs more than it saves.
__device__ __forceinline__ void tacg_pdl_prologue() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

template <typename... KArgs, typename... Args>
inline cudaError_t tacg_launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
                                   Args... args) {
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
// Static work split of the co-activation kernels: T items (layer-major) over `groups` CTA groups;
// group g owns items [g*T/groups, (g+1)*T/groups) and writes one scratch slot per layer it visits.
__host__ __device__ __forceinline__ long long group_lo(long long g, long long T, int groups) {
    if (T < (1ll << 24) && groups < 256) return (long long)(((unsigned)g * (unsigned)T) / (unsigned)groups);   // 32-bit divide
    return g * T / groups;
}

// the group that owns item x
__device__ __forceinline__ int group_of_item(long long x, long long T, int groups) {
    int g = (T < (1ll << 24) && groups < 256) ? (int)(((unsigned)x * (unsigned)groups) / (unsigned)T) : (int)((x * groups) / T);
    if (g >= groups) g = groups - 1;
    while (g + 1 < groups && group_lo(g + 1, T, groups) <= x) ++g;
    while (g > 0 && group_lo(g, T, groups) > x) --g;
    return g;
}


// Loads the KT expert ids of one token row.  KT in {2,4,6,8}: vector loads (the host
// checked the base alignment); KT == 0: k runtime, 2-byte loads.
template <int KT>
__device__ __forceinline__ void tacg_load_ids(const int16_t* __restrict__ row, int k, int (&e)[KT > 0 ? KT : 16]) {
    if constexpr (KT == 8) {
        const int4 v = __ldg(reinterpret_cast<const int4*>(row));
        e[0] = (short)(v.x & 0xffff); e[1] = v.x >> 16;
        e[2] = (short)(v.y & 0xffff); e[3] = v.y >> 16;
        e[4] = (short)(v.z & 0xffff); e[5] = v.z >> 16;
        e[6] = (short)(v.w & 0xffff); e[7] = v.w >> 16;
    } else if constexpr (KT == 6) {
        const int* p = reinterpret_cast<const int*>(row);
        const int a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2);
        e[0] = (short)(a & 0xffff); e[1] = a >> 16;
        e[2] = (short)(b & 0xffff); e[3] = b >> 16;
        e[4] = (short)(c & 0xffff); e[5] = c >> 16;
    } else if constexpr (KT == 4) {
        const int2 v = __ldg(reinterpret_cast<const int2*>(row));
        e[0] = (short)(v.x & 0xffff); e[1] = v.x >> 16;
        e[2] = (short)(v.y & 0xffff); e[3] = v.y >> 16;
    } else if constexpr (KT == 2) {
        const int a = __ldg(reinterpret_cast<const int*>(row));
        e[0] = (short)(a & 0xffff); e[1] = a >> 16;
    } else {
#pragma unroll
        for (int j = 0; j < 16; ++j) e[j] = (j < k) ? (int)__ldg(row + j) : -1;
    }
}

// The compile-time slot count for a (k, base pointer) pair; 0 = generic path.
static inline int tacg_pick_kt(int k, const void* base) {
    const uintptr_t a = reinterpret_cast<uintptr_t>(base);
    if ((k == 2 || k == 4 || k == 6 || k == 8) && (a % 16) == 0) return k;
    return 0;
}
#endif

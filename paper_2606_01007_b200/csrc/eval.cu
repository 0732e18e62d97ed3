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
#include <cooperative_groups.h>

#include "tacg_common.cuh"

namespace {

constexpr int kEvalThreads = 256;

struct LayerTables {        // per-layer lookup tables in shared memory
    unsigned short* info;   // [E] low byte = primary partition, high byte = number of valid replicas
    signed char* rep;       // [E*r] replica partitions, -1 = none
    double* S;              // [64] load snapshot
    unsigned long long feas;  // bit m = S[m] <= (1+theta)*mean(S)
};

// Step 4 of O10 for one token: serve[j] per slot (-1 = empty), returns the accessed set R.
template <int KT>
__device__ __forceinline__ unsigned long long
select_token(const int (&e)[KT > 0 ? KT : 16], int k, int E, int r, int home, const unsigned short* __restrict__ info,
             const signed char* __restrict__ rep, const double* __restrict__ S, unsigned long long feas,
             int (&sv)[KT > 0 ? KT : 16]) {
    constexpr int KM = KT > 0 ? KT : 16;
    unsigned long long R = 0ull;
    unsigned pending = 0u;
    // pass 1: experts with a single candidate are served by their primary regardless (Q18)
#pragma unroll
    for (int j = 0; j < KM; ++j) {
        sv[j] = -1;
        if (j < k && (unsigned)e[j] < (unsigned)E) {
            const unsigned in = info[e[j]];
            if ((in >> 8) == 0u) {
                sv[j] = (int)(in & 63u);
                R |= 1ull << (in & 63u);
            } else {
                pending |= 1u << j;
            }
        }
    }
    // pass 2: replicated experts in slot order; key (not local, snapshot load, candidate slot) (Q17)
    if (pending) {
#pragma unroll
        for (int j = 0; j < KM; ++j) {
            if (!((pending >> j) & 1u)) continue;
            const int ex = e[j];
            const int c0 = (int)(info[ex] & 63u);
            unsigned long long cmask = 1ull << c0;
            for (int a = 0; a < r; ++a) {
                const int c = rep[ex * r + a];
                if (c >= 0) cmask |= 1ull << (c & 63);
            }
            const bool anyfeas = (cmask & feas) != 0ull;       // else: fallback to all candidates
            int best = -1, bestloc = 0;
            double bestS = 0.0;
            for (int a = -1; a < r; ++a) {
                const int c = a < 0 ? c0 : (int)rep[ex * r + a];
                if (c < 0) continue;
                const int cm = c & 63;
                if (anyfeas && !((feas >> cm) & 1ull)) continue;
                const int nonlocal = (((R >> cm) & 1ull) || cm == home) ? 0 : 1;
                const double s = S[cm];
                if (best < 0 || nonlocal < bestloc || (nonlocal == bestloc && s < bestS)) {
                    best = cm; bestloc = nonlocal; bestS = s;
                }
            }
            sv[j] = best;
            R |= 1ull << best;
        }
    }
    return R;
}

__device__ __forceinline__ void load_tables(int E, int r, const int8_t* __restrict__ pr,
                                            const int8_t* __restrict__ rp, unsigned short* info, signed char* rep) {
    for (int e = threadIdx.x; e < E; e += blockDim.x) {
        unsigned n = 0;
        for (int a = 0; a < r; ++a) {
            const signed char c = rp[(size_t)e * r + a];
            rep[e * r + a] = c;
            n += (c >= 0) ? 1u : 0u;
        }
        info[e] = (unsigned short)(((unsigned)pr[e] & 63u) | (n << 8));
    }
}

// feas from a snapshot: mean summed left to right in double (Q19), theta widened from float.
__device__ __forceinline__ void load_guard(const double* S, int P, float theta, unsigned long long* feas_out) {
    // called by one thread
    double tot = 0.0;
    for (int m = 0; m < P; ++m) tot = __dadd_rn(tot, S[m]);
    const double Lbar = tot / (double)P;
    const double thr = __dmul_rn(__dadd_rn(1.0, (double)theta), Lbar);
    unsigned long long fm = 0ull;
    for (int m = 0; m < P; ++m)
        if (S[m] <= thr) fm |= 1ull << m;
    *feas_out = fm;
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
    unsigned char* cost;    // [L,N] or null
    signed char* serve;     // [L,N,k] or null
    unsigned long long* delta;   // scratch [L,nmb,P], zeroed before launch (only used when cpl > 1)
    unsigned* barrier;           // scratch [L], zeroed before launch
    int cpl;                // CTAs per layer
    int groups;             // number of concurrent layer groups = gridDim.x / cpl
};

template <int KT>
__global__ void __launch_bounds__(kEvalThreads)
eval_kernel(EvalParams p) {
    extern __shared__ unsigned char esm[];
    // layout: S[64] double | cnt[P][32] u32 | dsum[64] u64 | info[E] u16 | rep[E*r] i8
    double* S = reinterpret_cast<double*>(esm);
    unsigned* cnt = reinterpret_cast<unsigned*>(esm + 64 * sizeof(double));
    unsigned long long* dsum = reinterpret_cast<unsigned long long*>(cnt + (size_t)p.P * 32);
    unsigned short* info = reinterpret_cast<unsigned short*>(dsum + 64);
    signed char* rep = reinterpret_cast<signed char*>(info + ((p.E + 3) & ~3));
    __shared__ double Ls[64];              // EMA state of this layer
    __shared__ unsigned long long ltot[64];  // cumulative integer load of this layer
    __shared__ unsigned long long feas_s;
    __shared__ unsigned long long comm_s[16];

    const int group = blockIdx.x / p.cpl;
    const int part = blockIdx.x % p.cpl;
    if (group >= p.groups) return;
    const int lane = threadIdx.x & 31;
    const int P = p.P, k = p.k, E = p.E, F = p.F, r = p.r;

    for (int layer = group; layer < p.L; layer += p.groups) {
        __syncthreads();
        load_tables(E, r, p.primary + (size_t)layer * E, p.replicas ? p.replicas + (size_t)layer * E * r : nullptr,
                    info, rep);
        for (int i = threadIdx.x; i < P * 32; i += blockDim.x) cnt[i] = 0u;
        if (threadIdx.x < 64) {
            Ls[threadIdx.x] = (p.load_state && threadIdx.x < P) ? p.load_state[(size_t)layer * P + threadIdx.x] : 0.0;
            ltot[threadIdx.x] = 0ull;
        }
        if (threadIdx.x < 16) comm_s[threadIdx.x] = 0ull;
        __syncthreads();
        unsigned long long span_acc[8], rem_acc[8];   // lane 0 of each warp accumulates per family
#pragma unroll
        for (int f = 0; f < 8; ++f) { span_acc[f] = 0ull; rem_acc[f] = 0ull; }
        const int16_t* base = p.indices + (size_t)layer * (size_t)p.N * (size_t)k;

        for (long long mb = 0; mb < p.nmb; ++mb) {
            // steps 1-3: snapshot and guard
            if (threadIdx.x < 64) S[threadIdx.x] = Ls[threadIdx.x];
            __syncthreads();
            if (threadIdx.x == 0) load_guard(S, P, p.theta, &feas_s);
            __syncthreads();
            const unsigned long long feas = feas_s;
            // step 4: this CTA's slice of the micro-batch
            const long long mb_begin = mb * p.B;
            const long long mb_end = min(p.N, mb_begin + p.B);
            const long long len = mb_end - mb_begin;
            const long long per = ((len + p.cpl - 1) / p.cpl + 31) / 32 * 32;
            const long long t0 = mb_begin + (long long)part * per;
            const long long t1 = min(mb_end, t0 + per);
            for (long long tb = t0; tb < t1; tb += kEvalThreads) {
                const long long t = tb + threadIdx.x;
                int f = -1;
                if (t < t1) f = p.family[t];
                const bool live = (unsigned)f < (unsigned)F;
                int packed = 0;
                if (live) {
                    int e[KT > 0 ? KT : 16], sv[KT > 0 ? KT : 16];
                    tacg_load_ids<KT>(base + (size_t)t * k, k, e);
                    const int home = (int)((p.token_offset + t) % P);
                    const unsigned long long R = select_token<KT>(e, k, E, r, home, info, rep, S, feas, sv);
#pragma unroll
                    for (int j = 0; j < (KT > 0 ? KT : 16); ++j)
                        if (j < k && sv[j] >= 0) atomicAdd(&cnt[sv[j] * 32 + lane], 1u);
                    const int nR = __popcll(R);
                    const int rem = __popcll(R & ~(1ull << home));
                    packed = max(0, nR - 1) | (rem << 16);
                    if (p.cost) p.cost[(size_t)layer * p.N + t] = (unsigned char)rem;
                    if (p.serve) {
#pragma unroll
                        for (int j = 0; j < (KT > 0 ? KT : 16); ++j)
                            if (j < k) p.serve[((size_t)layer * p.N + t) * k + j] = (signed char)sv[j];
                    }
                } else if (t < t1) {
                    if (p.cost) p.cost[(size_t)layer * p.N + t] = 0;
                    if (p.serve)
                        for (int j = 0; j < k; ++j) p.serve[((size_t)layer * p.N + t) * k + j] = -1;
                }
                // per-family communication sums: one warp reduction per family (span | remote<<16)
#pragma unroll
                for (int g = 0; g < 8; ++g) {
                    if (g < F) {
                        const unsigned s = __reduce_add_sync(0xffffffffu, (unsigned)((live && f == g) ? packed : 0));
                        span_acc[g] += s & 0xffffu;
                        rem_acc[g] += s >> 16;
                    }
                }
            }
            // step 5: integer dispatch counts of the micro-batch, then Eq. 15
            __syncthreads();
            for (int m = threadIdx.x >> 5; m < P; m += kEvalThreads / 32) {
                const unsigned s = __reduce_add_sync(0xffffffffu, cnt[m * 32 + lane]);
                cnt[m * 32 + lane] = 0u;
                if (lane == 0) dsum[m] = (unsigned long long)s;
            }
            __syncthreads();
            if (p.cpl > 1) {
                unsigned long long* dl = p.delta + ((size_t)layer * p.nmb + mb) * P;
                if (threadIdx.x < P && dsum[threadIdx.x]) atomicAdd(&dl[threadIdx.x], dsum[threadIdx.x]);
                __threadfence();
                __syncthreads();
                if (threadIdx.x == 0) {
                    atomicAdd(&p.barrier[layer], 1u);
                    const unsigned target = (unsigned)((mb + 1) * p.cpl);
                    volatile unsigned* bar = p.barrier + layer;
                    while (*bar < target) __nanosleep(20);
                    __threadfence();
                }
                __syncthreads();
                if (threadIdx.x < P) dsum[threadIdx.x] = __ldcg(&dl[threadIdx.x]);
                __syncthreads();
            }
            if (threadIdx.x < P) {
                const unsigned long long d = dsum[threadIdx.x];
                Ls[threadIdx.x] = __dadd_rn(__dmul_rn(p.rho, Ls[threadIdx.x]), (double)d);   // no FMA (Q19)
                ltot[threadIdx.x] += d;
            }
            __syncthreads();
        }
        // layer epilogue: communication sums and, from part 0, loads and the final state
        if (lane == 0) {
#pragma unroll
            for (int g = 0; g < 8; ++g) {
                if (g < F) {
                    if (span_acc[g]) atomicAdd(&comm_s[g], span_acc[g]);
                    if (rem_acc[g]) atomicAdd(&comm_s[8 + g], rem_acc[g]);
                }
            }
        }
        __syncthreads();
        if (threadIdx.x < F) {
            if (comm_s[threadIdx.x]) atomicAdd(&p.comm_span[(size_t)layer * F + threadIdx.x], comm_s[threadIdx.x]);
            if (comm_s[8 + threadIdx.x]) atomicAdd(&p.comm_remote[(size_t)layer * F + threadIdx.x], comm_s[8 + threadIdx.x]);
        }
        if (part == 0 && threadIdx.x < P) {
            p.load[(size_t)layer * P + threadIdx.x] = ltot[threadIdx.x];
            if (p.load_state) p.load_state[(size_t)layer * P + threadIdx.x] = Ls[threadIdx.x];
        }
    }
}

// O11: (jain, maxvio, cv) per layer and for the loads summed over layers, fp64 -> fp32.
__global__ void fairness_kernel(const unsigned long long* __restrict__ load, int L, int P, float* __restrict__ out) {
    for (int row = blockIdx.x * blockDim.x + threadIdx.x; row <= L; row += gridDim.x * blockDim.x) {
        double tot = 0.0, sq = 0.0, mx = 0.0;
        for (int m = 0; m < P; ++m) {
            unsigned long long v = 0;
            if (row < L) v = load[(size_t)row * P + m];
            else for (int l = 0; l < L; ++l) v += load[(size_t)l * P + m];
            const double x = (double)v;
            tot += x; sq += x * x; mx = fmax(mx, x);
        }
        double jain = 1.0, maxvio = 0.0, cv = 0.0;
        if (tot != 0.0) {
            const double mean = tot / (double)P;
            double var = 0.0;
            for (int m = 0; m < P; ++m) {
                unsigned long long v = 0;
                if (row < L) v = load[(size_t)row * P + m];
                else for (int l = 0; l < L; ++l) v += load[(size_t)l * P + m];
                const double x = (double)v;
                var += (x - mean) * (x - mean);
            }
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
    extern __shared__ unsigned char ssm[];
    double* S = reinterpret_cast<double*>(ssm);
    unsigned short* info = reinterpret_cast<unsigned short*>(ssm + 64 * sizeof(double));
    signed char* rep = reinterpret_cast<signed char*>(info + ((E + 3) & ~3));
    __shared__ unsigned long long feas_s;
    const int layer = blockIdx.y;
    load_tables(E, r, primary + (size_t)layer * E, replicas ? replicas + (size_t)layer * E * r : nullptr, info, rep);
    if (threadIdx.x < 64) S[threadIdx.x] = threadIdx.x < P ? snapshot[(size_t)layer * P + threadIdx.x] : 0.0;
    __syncthreads();
    if (threadIdx.x == 0) load_guard(S, P, theta, &feas_s);
    __syncthreads();
    const unsigned long long feas = feas_s;
    const int16_t* base = indices + (size_t)layer * (size_t)N * (size_t)k;
    const long long stride = (long long)gridDim.x * kEvalThreads;
    for (long long t = (long long)blockIdx.x * kEvalThreads + threadIdx.x; t < N; t += stride) {
        int e[KT > 0 ? KT : 16], sv[KT > 0 ? KT : 16];
        tacg_load_ids<KT>(base + (size_t)t * k, k, e);
        const int home = (int)((token_offset + t) % P);
        select_token<KT>(e, k, E, r, home, info, rep, S, feas, sv);
        signed char* out = serve + ((size_t)layer * N + t) * k;
        if constexpr (KT == 8) {
            int2 v;
            v.x = (sv[0] & 0xff) | ((sv[1] & 0xff) << 8) | ((sv[2] & 0xff) << 16) | ((sv[3] & 0xff) << 24);
            v.y = (sv[4] & 0xff) | ((sv[5] & 0xff) << 8) | ((sv[6] & 0xff) << 16) | ((sv[7] & 0xff) << 24);
            *reinterpret_cast<int2*>(out) = v;
        } else {
#pragma unroll
            for (int j = 0; j < (KT > 0 ? KT : 16); ++j)
                if (j < k) out[j] = (signed char)sv[j];
        }
    }
}

size_t eval_smem_bytes(int E, int P, int r) {
    return 64 * sizeof(double) + sizeof(unsigned) * (size_t)P * 32 + 64 * sizeof(unsigned long long) +
           sizeof(unsigned short) * (size_t)((E + 3) & ~3) + (size_t)E * (r > 0 ? r : 1) + 16;
}

template <int KT>
int launch_eval_t(tacg_ctx* ctx, EvalParams& p) {
    const size_t smem = eval_smem_bytes(p.E, p.P, p.r);
    auto kern = eval_kernel<KT>;
    int occ = 0;
    TACG_CUDA_TRY(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, kEvalThreads, smem));
    if (occ < 1) occ = 1;
    const int max_grid = ctx->sm_count * occ;
    // CTAs per layer: spread the grid over the layers; never more CTAs than 32-token slices of a micro-batch
    long long cpl = max(1, max_grid / p.L);
    const long long slices = max(1ll, (min(p.B, p.N) + 2 * kEvalThreads - 1) / (2 * kEvalThreads));
    if (cpl > slices) cpl = slices;
    p.cpl = (int)cpl;
    p.groups = (int)min((long long)p.L, (long long)max_grid / cpl);
    const int grid = p.groups * p.cpl;
    const bool waits = p.cpl > 1 && p.nmb > 1;     // CTAs of a group meet at a barrier per micro-batch
    size_t off = 0;
    const size_t o_delta = off; off += tacg_align_up(sizeof(unsigned long long) * (size_t)p.L * (size_t)p.nmb * p.P, 256);
    const size_t o_bar = off;   off += tacg_align_up(sizeof(unsigned) * (size_t)p.L, 256);
    char* base = static_cast<char*>(tacg_scratch(ctx, off));
    if (!base) return TACG_ERR_CUDA;
    p.delta = reinterpret_cast<unsigned long long*>(base + o_delta);
    p.barrier = reinterpret_cast<unsigned*>(base + o_bar);
    if (p.cpl > 1) TACG_CUDA_TRY(ctx, cudaMemsetAsync(base, 0, off, ctx->stream));
    tacg_prof_scope prof(ctx, TACG_PROF_EVAL);
    if (waits) {
        void* args[] = {&p};
        TACG_CUDA_TRY(ctx, cudaLaunchCooperativeKernel((const void*)kern, dim3(grid), dim3(kEvalThreads), args, smem,
                                                       ctx->stream));
        ctx->launches += 1;
    } else {
        kern<<<grid, kEvalThreads, smem, ctx->stream>>>(p);
        TACG_LAUNCH_CHECK(ctx);
    }
    return TACG_OK;
}

template <int KT>
int launch_select_t(tacg_ctx* ctx, const int16_t* indices, int64_t N, int k, int L, int E, int P,
                    const int8_t* primary, const int8_t* replicas, int r, const double* snapshot, float theta,
                    int64_t token_offset, int8_t* serve) {
    const size_t smem = 64 * sizeof(double) + sizeof(unsigned short) * (size_t)((E + 3) & ~3) +
                        (size_t)E * (r > 0 ? r : 1) + 16;
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
                     uint64_t* comm_span, uint64_t* comm_remote, float* fairness, uint8_t* cost_per_token,
                     int8_t* serve) {
    TACG_CUDA_TRY(ctx, cudaMemsetAsync(comm_span, 0, sizeof(uint64_t) * (size_t)L * F, ctx->stream));
    TACG_CUDA_TRY(ctx, cudaMemsetAsync(comm_remote, 0, sizeof(uint64_t) * (size_t)L * F, ctx->stream));
    TACG_CUDA_TRY(ctx, cudaMemsetAsync(load, 0, sizeof(uint64_t) * (size_t)L * P, ctx->stream));
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
        p.cost = cost_per_token;
        p.serve = reinterpret_cast<signed char*>(serve);
        p.delta = nullptr; p.barrier = nullptr; p.cpl = 1; p.groups = 1;
        int rc;
        switch (tacg_pick_kt(k, indices)) {
            case 2: rc = launch_eval_t<2>(ctx, p); break;
            case 4: rc = launch_eval_t<4>(ctx, p); break;
            case 6: rc = launch_eval_t<6>(ctx, p); break;
            case 8: rc = launch_eval_t<8>(ctx, p); break;
            default: rc = launch_eval_t<0>(ctx, p); break;
        }
        if (rc != TACG_OK) return rc;
    }
    fairness_kernel<<<1, 64, 0, ctx->stream>>>(reinterpret_cast<const unsigned long long*>(load), L, P, fairness);
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

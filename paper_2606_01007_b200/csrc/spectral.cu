// Capacity-feasible expert grouping by the paper's spectral-then-repair procedure
// (Eq. 9-10).  An offline, latency-bound step: one CTA per
// layer walks the whole procedure in fp64 with the layer's E x E matrices resident in L2.
//
//   Stage 1  S = (W + W^T)/2 / max;  A = S + jitter*I;  deg = rowsum A;  Nrm = D^-1/2 A D^-1/2.
//            The M smallest eigenvectors of L_sym = I - Nrm are the M largest of B = I + Nrm, which
//            is positive semi-definite, so a one-sided (Hestenes) Jacobi iteration on the columns of
//            B converges to lambda_i * v_i: no second matrix for the eigenvectors, and every
//            rotation touches two contiguous columns.  One warp per column pair, the n/2 disjoint
//            pairs of a round-robin round run concurrently.  k-means (Lloyd, farthest-point start)
//            runs on the rows of the E x M embedding.
//   Stage 2  overfull groups keep their top-`capacity` members by intra-group affinity, the rest
//            are inserted greedily by Eq. 10.  Sums run in increasing expert id so that, given the
//            same Stage-1 labels, the result is the oracle's bit for bit.
// Readings Q33-Q37 of DESIGN.md fix what the text leaves open.
#include "tacg_common.cuh"

namespace {

constexpr int kThreads = 512;    // 32 column elements per lane live in registers during a rotation
constexpr int kWarps = kThreads / 32;
constexpr int kMaxPerLane = 16;   // E <= 512
constexpr int kMaxSweeps = 40;
constexpr double kRotTol = 5e-14; // |a_p . a_q| <= tol * |a_p||a_q| counts as orthogonal

struct SpectralParams {
    const float* W;            // [L,E,E]
    int E, P, capacity, iters;
    double jitter;
    const int8_t* labels_in;   // [L,E] or NULL
    int8_t* primary;           // [L,E]
    int8_t* labels0;           // [L,E] or NULL
    double* embed;             // [L,E,P] or NULL
    double* S;                 // scratch [L,E,E]
    double* B;                 // scratch [L,E,E], column c at B + c*E
    double* X;                 // scratch [L,E,P]
};

struct Shared {
    double red_v[kWarps];
    int red_i[kWarps];
    double bcast_v;
    int bcast_i;
    int flag;
    int pool_n;
};

// id of the largest v over the block; ties -> lower id.  Every thread calls it.
__device__ int block_argmax(double v, int id, Shared* sh) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double ov = __shfl_xor_sync(0xffffffffu, v, o);
        const int oi = __shfl_xor_sync(0xffffffffu, id, o);
        if (ov > v || (ov == v && oi < id)) { v = ov; id = oi; }
    }
    if (lane == 0) { sh->red_v[warp] = v; sh->red_i[warp] = id; }
    __syncthreads();
    if (warp == 0) {
        v = lane < kWarps ? sh->red_v[lane] : -INFINITY;
        id = lane < kWarps ? sh->red_i[lane] : 0x7fffffff;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, v, o);
            const int oi = __shfl_xor_sync(0xffffffffu, id, o);
            if (ov > v || (ov == v && oi < id)) { v = ov; id = oi; }
        }
        if (lane == 0) { sh->bcast_v = v; sh->bcast_i = id; }
    }
    __syncthreads();
    const int out = sh->bcast_i;
    __syncthreads();
    return out;
}

__device__ double block_max(double v, Shared* sh) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if (lane == 0) sh->red_v[warp] = v;
    __syncthreads();
    if (warp == 0) {
        v = lane < kWarps ? sh->red_v[lane] : -INFINITY;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
        if (lane == 0) sh->bcast_v = v;
    }
    __syncthreads();
    const double out = sh->bcast_v;
    __syncthreads();
    return out;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// One-sided Jacobi on the E columns of B until no pair needs a rotation.
__device__ void jacobi_columns(double* __restrict__ B, int E, Shared* sh) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int n = E + (E & 1);
    for (int sweep = 0; sweep < kMaxSweeps; ++sweep) {
        if (threadIdx.x == 0) sh->flag = 0;
        __syncthreads();
        for (int r = 0; r < n - 1; ++r) {
            for (int pi = warp; pi < n / 2; pi += kWarps) {
                int a, b;
                if (pi == 0) { a = r; b = n - 1; }
                else { a = (r + pi) % (n - 1); b = (r - pi + n - 1) % (n - 1); }
                if (a >= E || b >= E) continue;               // the phantom column of an odd E
                double* cp = B + (size_t)min(a, b) * E;
                double* cq = B + (size_t)max(a, b) * E;
                double xp[kMaxPerLane], xq[kMaxPerLane];
                double alpha = 0.0, beta = 0.0, gamma = 0.0;
#pragma unroll
                for (int t = 0; t < kMaxPerLane; ++t) {
                    const int i = lane + 32 * t;
                    xp[t] = (i < E) ? cp[i] : 0.0;
                    xq[t] = (i < E) ? cq[i] : 0.0;
                    alpha += xp[t] * xp[t];
                    beta += xq[t] * xq[t];
                    gamma += xp[t] * xq[t];
                }
                alpha = warp_sum(alpha);
                beta = warp_sum(beta);
                gamma = warp_sum(gamma);
                if (fabs(gamma) <= kRotTol * sqrt(alpha * beta)) continue;
                const double zeta = (beta - alpha) / (2.0 * gamma);
                const double t_ = copysign(1.0, zeta) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
                const double c = 1.0 / sqrt(1.0 + t_ * t_), s = c * t_;
#pragma unroll
                for (int t = 0; t < kMaxPerLane; ++t) {
                    const int i = lane + 32 * t;
                    if (i < E) {
                        cp[i] = c * xp[t] - s * xq[t];
                        cq[i] = s * xp[t] + c * xq[t];
                    }
                }
                if (lane == 0) sh->flag = 1;
            }
            __syncthreads();
        }
        const int any = sh->flag;
        __syncthreads();
        if (!any) break;
    }
}

__global__ void __launch_bounds__(kThreads) spectral_place_kernel(SpectralParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int E = p.E, M = p.P, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int l = blockIdx.x;
    Shared* sh = reinterpret_cast<Shared*>(smem_raw);
    double* deg = reinterpret_cast<double*>(smem_raw + 512);   // [E]   degree, later intra-group affinity
    double* val = deg + E;                                      // [E]   column norms, later min distance
    double* cent = val + E;                                     // [M*M] k-means centres
    int* labels = reinterpret_cast<int*>(cent + M * M);         // [E]
    int* sizes = labels + E;                                    // [M]
    int* pool = sizes + M;                                      // [E]
    int* mark = pool + E;                                       // [E]   column rank, later eviction marks

    const float* W = p.W + (size_t)l * E * E;
    double* S = p.S + (size_t)l * E * E;
    double* B = p.B + (size_t)l * E * E;
    double* X = p.X + (size_t)l * E * M;

    // ---- scaled symmetric affinity ----
    double mx = -INFINITY;
    for (int idx = tid; idx < E * E; idx += kThreads) {
        const int i = idx / E, j = idx - i * E;
        const double v = ((double)W[idx] + (double)W[j * E + i]) * 0.5;
        S[idx] = v;
        mx = fmax(mx, v);
    }
    const double top = block_max(mx, sh);
    if (top > 0.0)
        for (int idx = tid; idx < E * E; idx += kThreads) S[idx] = S[idx] / top;
    __syncthreads();

    if (p.labels_in) {
        for (int e = tid; e < E; e += kThreads) labels[e] = p.labels_in[(size_t)l * E + e];
        __syncthreads();
    } else {
        // ---- Stage 1: embedding ----
        for (int e = tid; e < E; e += kThreads) {
            double s = 0.0;
            for (int j = 0; j < E; ++j) s += S[(size_t)j * E + e];     // S is bitwise symmetric: column read, row sum
            deg[e] = s + p.jitter;
        }
        __syncthreads();
        for (int idx = tid; idx < E * E; idx += kThreads) {
            const int c = idx / E, i = idx - c * E;
            const double a = S[idx] + (i == c ? p.jitter : 0.0);
            B[idx] = (i == c ? 1.0 : 0.0) + a / (sqrt(deg[i]) * sqrt(deg[c]));
        }
        __syncthreads();
        jacobi_columns(B, E, sh);
        for (int c = warp; c < E; c += kWarps) {
            double s = 0.0;
            for (int i = lane; i < E; i += 32) s += B[(size_t)c * E + i] * B[(size_t)c * E + i];
            s = warp_sum(s);
            if (lane == 0) val[c] = sqrt(s);
        }
        __syncthreads();
        for (int c = tid; c < E; c += kThreads) {
            int rank = 0;
            for (int c2 = 0; c2 < E; ++c2) rank += (val[c2] > val[c]) || (val[c2] == val[c] && c2 < c);
            mark[c] = rank;
        }
        __syncthreads();
        for (int c = warp; c < E; c += kWarps) {
            const int rank = mark[c];
            if (rank >= M) continue;
            const double inv = val[c] > 0.0 ? 1.0 / val[c] : 0.0;
            for (int i = lane; i < E; i += 32) X[(size_t)i * M + rank] = B[(size_t)c * E + i] * inv;
        }
        __syncthreads();
        if (p.embed)
            for (int idx = tid; idx < E * M; idx += kThreads) p.embed[(size_t)l * E * M + idx] = X[idx];

        // ---- Stage 1: k-means, farthest-point start ----
        int first = 0;
        {
            double bv = -INFINITY;
            int bi = 0x7fffffff;
            for (int e = tid; e < E; e += kThreads)
                if (deg[e] > bv) { bv = deg[e]; bi = e; }
            first = block_argmax(bv, bi, sh);
        }
        for (int t = tid; t < M; t += kThreads) cent[t] = X[(size_t)first * M + t];
        for (int e = tid; e < E; e += kThreads) labels[e] = -1;
        __syncthreads();
        for (int e = tid; e < E; e += kThreads) {
            double d = 0.0;
            for (int t = 0; t < M; ++t) { const double u = X[(size_t)e * M + t] - cent[t]; d += u * u; }
            val[e] = d;
        }
        __syncthreads();
        for (int c = 1; c < M; ++c) {
            double bv = -INFINITY;
            int bi = 0x7fffffff;
            for (int e = tid; e < E; e += kThreads)
                if (val[e] > bv) { bv = val[e]; bi = e; }
            const int nxt = block_argmax(bv, bi, sh);
            for (int t = tid; t < M; t += kThreads) cent[c * M + t] = X[(size_t)nxt * M + t];
            __syncthreads();
            for (int e = tid; e < E; e += kThreads) {
                double d = 0.0;
                for (int t = 0; t < M; ++t) { const double u = X[(size_t)e * M + t] - cent[c * M + t]; d += u * u; }
                val[e] = fmin(val[e], d);
            }
            __syncthreads();
        }
        for (int it = 0; it < p.iters; ++it) {
            if (tid == 0) sh->flag = 0;
            __syncthreads();
            for (int e = tid; e < E; e += kThreads) {
                double bd = INFINITY;
                int bc = 0;
                for (int c = 0; c < M; ++c) {
                    double d = 0.0;
                    for (int t = 0; t < M; ++t) { const double u = X[(size_t)e * M + t] - cent[c * M + t]; d += u * u; }
                    if (d < bd) { bd = d; bc = c; }
                }
                if (bc != labels[e]) { labels[e] = bc; sh->flag = 1; }
            }
            __syncthreads();
            const int changed = sh->flag;
            __syncthreads();
            if (!changed) break;
            for (int ct = tid; ct < M * M; ct += kThreads) {
                const int c = ct / M, t = ct - c * M;
                double s = 0.0;
                int cnt = 0;
                for (int e = 0; e < E; ++e)
                    if (labels[e] == c) { s += X[(size_t)e * M + t]; ++cnt; }
                if (cnt) cent[ct] = s / (double)cnt;
            }
            __syncthreads();
        }
    }
    if (p.labels0)
        for (int e = tid; e < E; e += kThreads) p.labels0[(size_t)l * E + e] = (int8_t)labels[e];

    // ---- Stage 2: capacity repair ----
    for (int m = tid; m < M; m += kThreads) {
        int cnt = 0;
        for (int e = 0; e < E; ++e) cnt += labels[e] == m;
        sizes[m] = cnt;
    }
    for (int e = tid; e < E; e += kThreads) {
        const int m = labels[e];
        double s = 0.0;
        for (int e2 = 0; e2 < E; ++e2)
            if (e2 != e && labels[e2] == m) s += S[(size_t)e2 * E + e];
        deg[e] = s;
        mark[e] = 0;
    }
    if (tid == 0) sh->pool_n = 0;
    __syncthreads();
    for (int m = 0; m < M; ++m) {
        const int over = sizes[m] - p.capacity;
        if (over <= 0) continue;                               // uniform: sizes is shared
        const int base = sh->pool_n;
        for (int e = tid; e < E; e += kThreads) {
            if (labels[e] != m) continue;
            int rank = 0;
            for (int e2 = 0; e2 < E; ++e2)
                rank += labels[e2] == m && (deg[e2] > deg[e] || (deg[e2] == deg[e] && e2 < e));
            if (rank >= p.capacity) { pool[base + rank - p.capacity] = e; mark[e] = 1; }
        }
        __syncthreads();
        if (tid == 0) { sh->pool_n = base + over; sizes[m] = p.capacity; }
        __syncthreads();
    }
    for (int e = tid; e < E; e += kThreads)
        if (mark[e]) labels[e] = -1;
    __syncthreads();
    const int pool_n = sh->pool_n;
    for (int pi = 0; pi < pool_n; ++pi) {
        const int e = pool[pi];
        double inc = -INFINITY;
        int id = 0x7fffffff;
        if (tid < M && sizes[tid] < p.capacity) {              // Eq. 10: non-full groups only
            double s = 0.0;
            for (int e2 = 0; e2 < E; ++e2)
                if (labels[e2] == tid) s += S[(size_t)e2 * E + e];
            inc = s;
            id = tid;
        }
        const int best = block_argmax(inc, id, sh);
        if (tid == 0) { labels[e] = best; sizes[best] += 1; }
        __syncthreads();
    }
    for (int e = tid; e < E; e += kThreads) p.primary[(size_t)l * E + e] = (int8_t)labels[e];
}

}  // namespace

int tacg_launch_spectral(tacg_ctx* ctx, const float* W, int L, int E, int P, int capacity, double jitter, int iters,
                         const int8_t* labels_in, int8_t* primary, int8_t* labels0, double* embed) {
    const size_t mat = tacg_align_up((size_t)L * E * E * sizeof(double), 256);
    const size_t emb = tacg_align_up((size_t)L * E * P * sizeof(double), 256);
    unsigned char* base = static_cast<unsigned char*>(tacg_scratch(ctx, 2 * mat + emb));
    if (!base) return TACG_ERR_CUDA;
    SpectralParams p;
    p.W = W; p.E = E; p.P = P; p.capacity = capacity; p.iters = iters; p.jitter = jitter;
    p.labels_in = labels_in; p.primary = primary; p.labels0 = labels0; p.embed = embed;
    p.S = reinterpret_cast<double*>(base);
    p.B = reinterpret_cast<double*>(base + mat);
    p.X = reinterpret_cast<double*>(base + 2 * mat);
    const size_t smem = 512 + sizeof(double) * ((size_t)2 * E + (size_t)P * P) + sizeof(int) * ((size_t)3 * E + P);
    static_assert(sizeof(Shared) <= 512, "Shared must fit its slot");
    TACG_CUDA_TRY(ctx, cudaFuncSetAttribute(spectral_place_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    spectral_place_kernel<<<L, kThreads, smem, ctx->stream>>>(p);
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

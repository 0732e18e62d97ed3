/* tacg.h -- C ABI of libtacg: the data-parallel hot path behind TACG/GESR expert
 * placement (arxiv/paper_2606_01007), hand-written CUDA for sm_100a (B200).
 *
 * Citations are PAPER.md:<line> (the paper text) and SURVEY.md section 8; the
 * readings Q1..Q39 taken where the paper is silent are listed in DESIGN.md section 3.
 *
 * Conventions (all entry points)
 *   - Every pointer marked "dev" is DEVICE memory owned and allocated by the
 *     caller (e.g. a torch tensor's data_ptr()); the library never frees it and
 *     keeps no pointer after the call returns.  Scalars are passed by value.
 *   - Calls enqueue work on the ctx stream and return; outputs are valid after
 *     the caller synchronises that stream.  TACG_VALIDATE forces one
 *     synchronisation because it reads back an error word.
 *   - Return value: TACG_OK (0) or a negative tacg_status.  No error other than
 *     TACG_ERR_CUDA leaves an output partially written: shape / NULL errors are
 *     detected on the host before any launch.
 *   - Layouts are dense row-major with the last index fastest.
 *   - Limits: 1 <= k <= 16, 1 <= E <= 512, 1 <= P <= 64, 1 <= F <= 8,
 *     0 <= r <= 8, L >= 1, N >= 0.  Counts are uint32 (one C entry overflows
 *     only after 2^32 co-occurrences; documented, not checked).
 *   - Preconditions when not validating: the expert ids of one token are
 *     distinct (top-k without replacement).  A negative expert
 *     id is an empty slot (skipped); a negative family is a padding token
 *     (skipped).  Behaviour on duplicate ids is undefined without TACG_VALIDATE.
 *
 * There is no CPU fallback anywhere in this library: a call on a machine
 * without an sm_100 device fails with TACG_ERR_ARCH / TACG_ERR_CUDA.
 */
#ifndef TACG_H_
#define TACG_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum tacg_status {
    TACG_OK = 0,
    TACG_ERR_NULL = -1,      /* a required pointer is NULL */
    TACG_ERR_SHAPE = -2,     /* a size is outside the limits above, or E > P*capacity */
    TACG_ERR_BAD_INDEX = -3, /* TACG_VALIDATE only: expert id >= E, duplicate id in a token, family >= F */
    TACG_ERR_PLACEMENT = -4, /* TACG_VALIDATE only: primary outside [0,P), partition over capacity,
                                replica outside [-1,P), equal to the primary or duplicated */
    TACG_ERR_CUDA = -5,      /* a CUDA runtime call failed; text via tacg_last_detail */
    TACG_ERR_ARCH = -6       /* the device is not compute capability 10.x */
} tacg_status;

/* flags of tacg_coact_accumulate */
#define TACG_ZERO_FIRST 0x1u /* zero D, C and ntok on the stream before accumulating */
#define TACG_VALIDATE   0x2u /* check indices / family (coact) or primary / replicas (eval, select) on device */
#define TACG_PATH_AUTO  0x00u /* pick the co-activation kernel by shape (DESIGN.md 5.2 "Path choice") */
#define TACG_PATH_HIST  0x10u /* force the shared-memory / global atomic histogram kernel */
#define TACG_PATH_MMA   0x20u /* force the tcgen05 kind::i8 X^T X kernel; TACG_ERR_SHAPE if the shape is unsupported */
#define TACG_PATH_MASK  0x30u

typedef struct tacg_ctx tacg_ctx; /* opaque: device id, stream, scratch buffers, last error text */

/* Create a context on `device` bound to `cuda_stream` (a cudaStream_t, or NULL for
 * the legacy default stream).  Fails with TACG_ERR_ARCH unless the device is sm_100. */
int tacg_create(tacg_ctx** out, int device, void* cuda_stream);
int tacg_destroy(tacg_ctx* ctx);
/* Static description of a status code; never freed. */
const char* tacg_strerror(int code);
/* Copies the detail text of the last failing call on ctx (cudaGetErrorString text,
 * or "layer l token t ..." for validation) into buf (NUL-terminated, at most n bytes). */
int tacg_last_detail(tacg_ctx* ctx, char* buf, size_t n);
/* Which co-activation kernel the last tacg_coact_accumulate on ctx ran:
 * TACG_PATH_HIST or TACG_PATH_MMA (0 before the first call). */
int tacg_last_path(tacg_ctx* ctx);
/* Number of kernel launches the library has enqueued on ctx since creation. */
int64_t tacg_launch_count(tacg_ctx* ctx);
/* Library version, "major.minor". */
const char* tacg_version(void);

/* Optional device timing of the library's own kernels (used by bench.py for the roofline
 * figure): while enabled, every launch of the slot's kernel(s) is bracketed by CUDA events
 * on the ctx stream.  tacg_profile_read synchronises those events, returns the summed
 * duration in milliseconds and the number of bracketed launches since the last read, and
 * resets the slot.  Timing is off by default and costs nothing when off. */
#define TACG_PROF_COACT    0 /* the co-activation kernel (histogram or tcgen05), one launch per call */
#define TACG_PROF_AFFINITY 1 /* the kernels of tacg_affinity_swapgain, bracketed as one group per call */
#define TACG_PROF_EVAL     2 /* eval_kernel, one launch per call */
#define TACG_PROF_SLOTS    3
int tacg_profile_enable(tacg_ctx* ctx, int on);
int tacg_profile_read(tacg_ctx* ctx, int slot, double* total_ms, int64_t* launches);

/* Measured denominators for the roofline figures (the int8 tensor peak and the
 * shared-memory atomic peak are not in MEASURED_PEAKS.json, so the library measures them): runs a
 * micro-benchmark on every SM of the ctx device (one CTA per SM, a few milliseconds, synchronises the
 * ctx stream) and returns the throughput per second and per clock and SM (from the kernel's own cycle
 * counter).  Units: increments for the two atomic cases, integer operations (2 per multiply-add) for
 * the tensor case.  `which` outside the list: TACG_ERR_SHAPE. */
#define TACG_PEAK_ATOMS_SPREAD 0 /* shared-memory atomic increments, the 32 lanes of a warp on 32 different banks */
#define TACG_PEAK_ATOMS_RANDOM 1 /* shared-memory atomic increments on uniformly random words of a 128 KB table */
#define TACG_PEAK_I8_TENSOR    2 /* tcgen05.mma kind::i8, M=128 N=256 K=32, back to back, s32 accumulator in TMEM */
int tacg_measure_peak(tacg_ctx* ctx, int which, double* per_second, double* per_clk_sm);

/* S1+S2 -- per-family usage and co-activation counts
 * ("usage vector u ... coactivation matrix A ... frequency of expert pairs selected
 * by the same token", per layer and task family).
 *   for every layer l, token t with f = family[t] >= 0, expert set T = {indices[l,t,*] >= 0}:
 *     D[l,f,e] += 1 for e in T;  C[l,f,i,j] += 1 and C[l,f,j,i] += 1 for every unordered
 *     pair {i,j} of T;  C[l,f,e,e] is never touched;  ntok[f] += 1 once per token.
 * All three outputs ACCUMULATE (+=) so a long trace can be streamed in chunks;
 * TACG_ZERO_FIRST clears them first.  Integer results, bit-exact. */
int tacg_coact_accumulate(tacg_ctx* ctx,
                          const int16_t* indices, /* dev [L,N,k] expert ids of each token, per layer */
                          const int8_t* family,   /* dev [N] task family of each token, shared by all layers */
                          int64_t N, int k, int L, int E, int F,
                          uint32_t* D,            /* dev [L,F,E]   in/out */
                          uint32_t* C,            /* dev [L,F,E,E] in/out, symmetric, zero diagonal */
                          uint64_t* ntok,         /* dev [F]       in/out tokens per family */
                          uint32_t flags);

/* S3..S7 -- preferences (Eq. 2-6), task-modulated graph W = A-tilde
 * (Eq. 7-8), expert->partition affinity (inner sum of Eq. 10,
 * PAPER.md:121) and all-pairs swap gains (the "only if it improves" quantity of
 * PAPER.md:124 for every pair, north_star):
 *   u = D/sum_e D;  A^f = C^f/max(1,ntok[f]);  c = rowsum|A^f|;  dx = x^f - mean_{f'!=f} x^f';
 *   z = (dx-mu)/(sigma+eps) over experts (population sigma);  s = z(du)+z(dc);
 *   pref[e,:] = softmax_f(s/tau);  Abar = mean_f A^f;  Ahat = Abar/max Abar;
 *   W = (1-alpha) Ahat + alpha (pref pref^T) .* Ahat;  aff[e,m] = sum_{e': primary[e']=m} W[e,e'];
 *   gain[i,j] = aff[i,b]+aff[j,a]-aff[i,a]-aff[j,b]-2W[i,j] (a=primary[i] != b=primary[j]), else 0.
 * Computed in fp64 on device, stored as fp32.  Any output pointer may be NULL
 * (skipped).  primary may be NULL when aff and gain are NULL.  P and capacity are
 * checked (E <= P*capacity) when primary is given. */
int tacg_affinity_swapgain(tacg_ctx* ctx,
                           const uint32_t* D,    /* dev [L,F,E] */
                           const uint32_t* C,    /* dev [L,F,E,E] */
                           const uint64_t* ntok, /* dev [F] */
                           int L, int E, int F, int P, int capacity,
                           const int8_t* primary, /* dev [L,E] partition of each expert, or NULL */
                           float alpha, float tau, float eps,
                           float* pref,           /* dev [L,E,F] or NULL */
                           float* W,              /* dev [L,E,E] or NULL */
                           float* aff,            /* dev [L,E,P] or NULL */
                           float* gain);          /* dev [L,E,E] or NULL */

/* S8 -- GESR serving selection for ONE given load snapshot (Eq. 13-14 and the
 * fallback; pick rule Q17/Q18 of DESIGN.md):
 *   feas[m] = S[m] <= (1+theta) * mean(S);  experts without replicas are served by their
 *   primary (pass 1, they form the accessed set R);  each replicated expert, in slot order,
 *   picks among its feasible candidates (all candidates if none is feasible) the one
 *   minimising (not in R u {home}, S[c], candidate slot), and joins R.
 *   home = (token_offset + t) mod P.   serve[l,t,j] = -1 for an empty slot.
 * replicas may be NULL (or r = 0): serve = primary[indices]. */
int gesr_select(tacg_ctx* ctx,
                const int16_t* indices, /* dev [L,N,k] */
                int64_t N, int k, int L, int E, int P,
                const int8_t* primary,  /* dev [L,E] */
                const int8_t* replicas, /* dev [L,E,r], -1 = none; or NULL */
                int r,
                const double* load_snapshot, /* dev [L,P] */
                float theta, int64_t token_offset,
                int8_t* serve,          /* dev [L,N,k] out */
                uint32_t flags);        /* 0 or TACG_VALIDATE */

/* SURVEY.md 8(f) f2 (adjacent to the hot path) -- GESR offline step on the device: the generic-expert
 * score of Eq. 11 and the replica table of Eq. 12:
 *   A^f = C^f/max(1,ntok[f]);  Abar = mean_f A^f;  Cent[e] = sum_e' Abar[e,e'];
 *   Cons[e] = mean_f cos(A^f[e,:], Abar[e,:])  (0 when either vector is zero);
 *   Spec[e] = max_f ||A^f[e,:] - Abar[e,:]||_2;   score = Cent + lambda1*Cons - lambda2*Spec;
 *   per layer the n_rep experts of largest score (ties -> lower id) receive the r non-primary
 *   partitions of largest affinity aff[e,m] (aff as in tacg_affinity_swapgain with the same
 *   alpha, tau, eps and primary; ties -> lower id); replicas = -1 for every other expert and for
 *   slots beyond the P-1 other partitions.
 * fp64 on device; terms (optional) is stored as fp32.  Errors as tacg_affinity_swapgain, plus
 * TACG_ERR_SHAPE for n_rep < 0, r < 1 or r > 8. */
int gesr_build_replicas(tacg_ctx* ctx,
                        const uint32_t* D,     /* dev [L,F,E] */
                        const uint32_t* C,     /* dev [L,F,E,E] */
                        const uint64_t* ntok,  /* dev [F] */
                        int L, int E, int F, int P, int capacity,
                        const int8_t* primary, /* dev [L,E] */
                        float alpha, float tau, float eps,
                        float lambda1, float lambda2, int n_rep, int r,
                        int8_t* replicas,      /* dev [L,E,r] out */
                        float* terms);         /* dev [L,E,4] out or NULL: (score, Cent, Cons, Spec) */

/* SURVEY.md 8(f) f1 (adjacent to the hot path) -- capacity-feasible expert grouping by the
 * spectral-then-repair procedure of PAPER.md:110-124 (Eq. 9-10), per layer, on the device:
 *   Stage 1  S = (W + W^T)/2 divided by its largest entry;  A = S + jitter*I;  deg = rowsum A;
 *            L_sym = I - D^-1/2 A D^-1/2;  X = eigenvectors of its P smallest eigenvalues (rows not
 *            renormalised);  Lloyd's k-means with k = P on the rows of X from a farthest-point start
 *            (first centre = expert of largest degree), at most kmeans_iters rounds, an empty cluster
 *            keeps its centre, ties -> lower id.
 *   Stage 2  every group over `capacity` keeps its `capacity` members of largest intra-group
 *            affinity sum_{e' in group, e' != e} S[e,e'] (ties -> lower id); the others, group by
 *            group, strongest first, go to the non-full group of largest sum_{e' in group} S[e,e']
 *            (Eq. 10; ties -> lower group).
 * W must be non-negative.  labels_in (optional) replaces Stage 1: the repair alone, which is then
 * exact (sums in increasing expert id, fp64).  labels0 (optional) receives the Stage-1 labels and
 * embed (optional) the embedding; an eigenvector's sign and the basis inside a repeated eigenvalue
 * are not unique, the labels do not depend on them.  TACG_ERR_SHAPE for E > 512, P > min(64, E),
 * E > P*capacity, jitter <= 0 (with jitter = 0 an expert that never co-activates would have degree 0 and
 * D^-1/2 would not exist) or kmeans_iters < 1. */
int tacg_spectral_place(tacg_ctx* ctx,
                        const float* W,          /* dev [L,E,E] graph of tacg_affinity_swapgain */
                        int L, int E, int P, int capacity,
                        double jitter, int kmeans_iters,
                        const int8_t* labels_in, /* dev [L,E] in [0,P), or NULL */
                        int8_t* primary,         /* dev [L,E] out */
                        int8_t* labels0,         /* dev [L,E] out or NULL */
                        double* embed);          /* dev [L,E,P] out or NULL */

/* SURVEY.md 8(f) f3 (adjacent to the hot path) -- the motivation diagnostics of PAPER.md:469 from
 * the counts of tacg_coact_accumulate:
 *   P_f[l,e] = D[l,f,e]/max(1,ntok[f]);   frob[l,f,g] = ||P_f[l,:] - P_g[l,:]||_2 for l < L and
 *   frob[L,f,g] = ||P_f - P_g||_F over the whole [L,E] matrix;
 *   T_f[l] = the topk unordered pairs {i<j} of largest C[l,f,i,j] among pairs with a positive count
 *   (ties -> smaller (i,j));   jaccard[l,f,g] = |T_f ^ T_g| / |T_f u T_g| (0 when both are empty),
 *   jaccard[L,f,g] = mean over layers.
 * The sets are exact (integer select); the two outputs are fp64 on the device, stored as fp32.
 * TACG_ERR_SHAPE for E > 512, F > 8 or topk outside [1,256]. */
int tacg_family_divergence(tacg_ctx* ctx,
                           const uint32_t* D,    /* dev [L,F,E] */
                           const uint32_t* C,    /* dev [L,F,E,E] */
                           const uint64_t* ntok, /* dev [F] */
                           int L, int E, int F, int topk,
                           float* frob,          /* dev [L+1,F,F] out */
                           float* jaccard);      /* dev [L+1,F,F] out */

/* S8..S12 -- score a placement over a held-out trace (Eq. 13-15,
 * Comm per PAPER.md:363, Jain/MaxVio Eq. 17-18).  Tokens are processed
 * in micro-batches of `microbatch` consecutive tokens; every token of a micro-batch sees
 * the load state left by the previous micro-batch (north_star), then
 * state[m] = rho*state[m] + delta[m] (one rounded multiply, one rounded add, double).
 * With replicas == NULL or r == 0 the result does not depend on microbatch/theta/rho.
 * Outputs are OVERWRITTEN.  Integer outputs are bit-exact; fairness is computed in
 * fp64 and stored as fp32. */
int tacg_eval_placement(tacg_ctx* ctx,
                        const int16_t* indices, /* dev [L,N,k] */
                        const int8_t* family,   /* dev [N] */
                        int64_t N, int k, int L, int E, int F, int P,
                        const int8_t* primary,  /* dev [L,E] */
                        const int8_t* replicas, /* dev [L,E,r] or NULL */
                        int r, float theta, double rho,
                        int64_t microbatch,     /* B tokens; <= 0 or no replicas: one batch */
                        int64_t token_offset,   /* home = (token_offset + t) mod P */
                        double* load_state,     /* dev [L,P] in/out EMA state; NULL = start from 0, discard */
                        uint64_t* load,         /* dev [L,P] out dispatches served per partition */
                        uint64_t* comm_span,    /* dev [L,F] out sum over tokens of max(0,|cards|-1) */
                        uint64_t* comm_remote,  /* dev [L,F] out sum over tokens of |cards \ {home}| */
                        uint64_t* ntok,         /* dev [F]   out tokens per family */
                        float* fairness,        /* dev [L+1,3] out (jain, maxvio, cv); row L = loads summed over layers */
                        uint8_t* cost_per_token,/* dev [L,N] out |cards \ {home}| per token, or NULL */
                        int8_t* serve,          /* dev [L,N,k] out serving partition per slot, or NULL */
                        uint32_t flags);        /* 0 or TACG_VALIDATE */

/* The same evaluation for a placement WITHOUT replicas (S8, S9, S11, S12 of PAPER.md:145-159, 363, 453-463 with every
 * slot served by its primary partition), for callers that must not allocate: code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc.  It calls no cudaMalloc, cudaFree or allocating library routine
 * and does not touch the context's growable scratch: its only scratch, the per-slice partial sums
 * L * ceil(N / slice) * align4(P + 3F + 2) 32-bit words (slice <= 32768 tokens, chosen for the balance of the scan grid), lives in
 * a fixed device array of TACG_NOALLOC_SCRATCH_BYTES that every GPU holding the library keeps until the process
 * exits.  A call that needs more fails with TACG_ERR_SHAPE and a text naming the two sizes (nothing is launched);
 * split the layers over several calls, or use tacg_eval_placement.
 * Arguments, layouts and results are those of tacg_eval_placement with replicas = NULL (same kernels, same bits;
 * theta and microbatch do not enter without replicas); N >= 1; no TACG_VALIDATE; not bracketed by the profile events
 * of tacg_profile_enable.  EVERY call on a device shares the one array, which keeps the previous call's contents
 * (each call overwrites every word it later reads, nothing has to be cleared): two calls that overlap on the GPU
 * -- other streams, other contexts, other host threads -- race; the caller keeps them in order.
 * tacg_eval_primary_noalloc_prepare looks up the array's device address for the context's device (once per device;
 * the first tacg_eval_primary_noalloc on a device does the same): call it before a graph capture begins. */
#define TACG_NOALLOC_SCRATCH_BYTES (8u << 20)
int tacg_eval_primary_noalloc_prepare(tacg_ctx* ctx);
int tacg_eval_primary_noalloc(tacg_ctx* ctx,
                              const int16_t* indices, /* dev [L,N,k] */
                              const int8_t* family,   /* dev [N] */
                              int64_t N, int k, int L, int E, int F, int P,
                              const int8_t* primary,  /* dev [L,E] */
                              double rho,
                              int64_t token_offset,
                              double* load_state,     /* dev [L,P] in/out or NULL */
                              uint64_t* load,         /* dev [L,P] out */
                              uint64_t* comm_span,    /* dev [L,F] out */
                              uint64_t* comm_remote,  /* dev [L,F] out */
                              uint64_t* ntok,         /* dev [F]   out */
                              float* fairness,        /* dev [L+1,3] out */
                              uint8_t* cost_per_token,/* dev [L,N] out or NULL */
                              int8_t* serve);         /* dev [L,N,k] out or NULL */

#ifdef __cplusplus
}
#endif
#endif /* TACG_H_ */

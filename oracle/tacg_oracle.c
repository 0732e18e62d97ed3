/* ORACLE (full-size form) -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain C, loops, integers and fp64; written from /root/reference/PAPER.md
 * (cited as PAPER.md:<line>) with the readings Q1..Q28 of SURVEY.md 8(c),
 * restated in DESIGN.md "Readings".  It follows the same steps O1..O11, in
 * the same order, as oracle/ref.py (the definitional Python form), which pins
 * it on small inputs (tests/test_oracle_c.py).  It shares no code, header,
 * table or helper with paper_2606_01007_b200/csrc (the CUDA path).
 *
 * Used only by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs.  Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC
 * (-ffp-contract=off: Eq. 15 is one rounded multiply then one rounded add, Q19).
 * OpenMP, when enabled, only distributes whole layers (layers are independent
 * problems, Q22); there is no blocking, privatisation or reordering.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int orc_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* O1 -- counts.  PAPER.md:71.  D[L,F,E], C[L,F,E,E] and ntok[F] are accumulated (+=). */
int orc_coact(const int16_t* indices, const int8_t* family, int64_t N, int k, int L, int E, int F,
              uint32_t* D, uint32_t* C, uint64_t* ntok) {
    for (int64_t t = 0; t < N; ++t) {
        int f = family[t];
        if (f >= 0 && f < F) ntok[f] += 1;
    }
#pragma omp parallel for schedule(dynamic, 1)
    for (int l = 0; l < L; ++l) {
        const int16_t* idx = indices + (size_t)l * (size_t)N * (size_t)k;
        uint32_t* Dl = D + (size_t)l * F * E;
        uint32_t* Cl = C + (size_t)l * F * E * E;
        for (int64_t t = 0; t < N; ++t) {
            int f = family[t];
            if (f < 0 || f >= F) continue;
            const int16_t* T = idx + (size_t)t * k;
            for (int a = 0; a < k; ++a) {
                int i = T[a];
                if (i < 0) continue;
                Dl[(size_t)f * E + i] += 1;
                for (int b = a + 1; b < k; ++b) {
                    int j = T[b];
                    if (j < 0 || j == i) continue;      /* C[l,f,e,e] is never touched */
                    Cl[((size_t)f * E + i) * E + j] += 1;
                    Cl[((size_t)f * E + j) * E + i] += 1;
                }
            }
        }
    }
    return 0;
}

/* Eq. 4, population sigma (Q6). */
static void zscore(const double* x, int E, double eps, double* z) {
    double mu = 0.0;
    for (int e = 0; e < E; ++e) mu += x[e];
    mu /= E;
    double var = 0.0;
    for (int e = 0; e < E; ++e) var += (x[e] - mu) * (x[e] - mu);
    var /= E;
    double sigma = sqrt(var);
    for (int e = 0; e < E; ++e) z[e] = (x[e] - mu) / (sigma + eps);
}

/* O2..O8 -- preferences (Eq. 2-6), graph (Eq. 7-8), affinity (Eq. 10), swap gains.
 * Outputs are fp64: pref[L,E,F], W[L,E,E], aff[L,E,P], gain[L,E,E]; any may be NULL. */
int orc_affinity_swapgain(const uint32_t* D, const uint32_t* C, const uint64_t* ntok,
                          int L, int E, int F, int P, const int8_t* primary,
                          double alpha, double tau, double eps,
                          double* pref_out, double* W_out, double* aff_out, double* gain_out) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int l = 0; l < L; ++l) {
        const uint32_t* Dl = D + (size_t)l * F * E;
        const uint32_t* Cl = C + (size_t)l * F * E * E;
        double* u = (double*)calloc((size_t)F * E, sizeof(double));
        double* c = (double*)calloc((size_t)F * E, sizeof(double));
        double* dx = (double*)calloc((size_t)E, sizeof(double));
        double* zu = (double*)calloc((size_t)F * E, sizeof(double));
        double* zc = (double*)calloc((size_t)F * E, sizeof(double));
        double* pref = (double*)calloc((size_t)E * F, sizeof(double));
        double* Ahat = (double*)calloc((size_t)E * E, sizeof(double));
        double* W = (double*)calloc((size_t)E * E, sizeof(double));
        double* aff = (double*)calloc((size_t)E * P, sizeof(double));
        /* O2 */
        for (int f = 0; f < F; ++f) {
            uint64_t tot = 0;
            for (int e = 0; e < E; ++e) tot += Dl[(size_t)f * E + e];
            double dtot = (double)(tot > 0 ? tot : 1);
            double nf = (double)(ntok[f] > 0 ? ntok[f] : 1);
            for (int e = 0; e < E; ++e) {
                u[(size_t)f * E + e] = (double)Dl[(size_t)f * E + e] / dtot;
                double s = 0.0;
                for (int e2 = 0; e2 < E; ++e2) s += fabs((double)Cl[((size_t)f * E + e) * E + e2] / nf);
                c[(size_t)f * E + e] = s;
            }
        }
        /* O3, O4 */
        for (int f = 0; f < F; ++f) {
            for (int pass = 0; pass < 2; ++pass) {
                const double* x = pass == 0 ? u : c;
                for (int e = 0; e < E; ++e) {
                    double other = 0.0;
                    if (F > 1) {
                        for (int g = 0; g < F; ++g) if (g != f) other += x[(size_t)g * E + e];
                        other /= (double)(F - 1);
                    }
                    dx[e] = x[(size_t)f * E + e] - other;
                }
                zscore(dx, E, eps, (pass == 0 ? zu : zc) + (size_t)f * E);
            }
        }
        /* O5 */
        for (int e = 0; e < E; ++e) {
            double m = -INFINITY;
            for (int f = 0; f < F; ++f) {
                double s = (zu[(size_t)f * E + e] + zc[(size_t)f * E + e]) / tau;
                if (s > m) m = s;
            }
            double tot = 0.0;
            for (int f = 0; f < F; ++f) {
                double s = (zu[(size_t)f * E + e] + zc[(size_t)f * E + e]) / tau;
                pref[(size_t)e * F + f] = exp(s - m);
                tot += pref[(size_t)e * F + f];
            }
            for (int f = 0; f < F; ++f) pref[(size_t)e * F + f] /= tot;
        }
        /* O6 */
        double mx = 0.0;
        for (int i = 0; i < E; ++i)
            for (int j = 0; j < E; ++j) {
                double s = 0.0;
                for (int f = 0; f < F; ++f) {
                    double nf = (double)(ntok[f] > 0 ? ntok[f] : 1);
                    s += (double)Cl[((size_t)f * E + i) * E + j] / nf;
                }
                s /= (double)F;
                Ahat[(size_t)i * E + j] = s;
                if (s > mx) mx = s;
            }
        for (int i = 0; i < E; ++i)
            for (int j = 0; j < E; ++j) {
                double ah = mx > 0.0 ? Ahat[(size_t)i * E + j] / mx : 0.0;
                double at = 0.0;
                for (int f = 0; f < F; ++f) at += pref[(size_t)i * F + f] * pref[(size_t)j * F + f];
                W[(size_t)i * E + j] = (1.0 - alpha) * ah + alpha * (at * ah);
            }
        /* O7 */
        if (primary) {
            const int8_t* pr = primary + (size_t)l * E;
            for (int e = 0; e < E; ++e)
                for (int e2 = 0; e2 < E; ++e2) aff[(size_t)e * P + pr[e2]] += W[(size_t)e * E + e2];
            /* O8 */
            if (gain_out) {
                double* G = gain_out + (size_t)l * E * E;
                for (int i = 0; i < E; ++i)
                    for (int j = 0; j < E; ++j) {
                        int a = pr[i], b = pr[j];
                        G[(size_t)i * E + j] = (a == b) ? 0.0
                            : aff[(size_t)i * P + b] + aff[(size_t)j * P + a] - aff[(size_t)i * P + a]
                              - aff[(size_t)j * P + b] - 2.0 * W[(size_t)i * E + j];
                    }
            }
        }
        if (pref_out) memcpy(pref_out + (size_t)l * E * F, pref, sizeof(double) * E * F);
        if (W_out) memcpy(W_out + (size_t)l * E * E, W, sizeof(double) * E * E);
        if (aff_out) memcpy(aff_out + (size_t)l * E * P, aff, sizeof(double) * E * P);
        free(u); free(c); free(dx); free(zu); free(zc); free(pref); free(Ahat); free(W); free(aff);
    }
    return 0;
}

/* Eq. 13-14: feas[m] = S[m] <= (1+theta) * Lbar, Lbar summed left to right. */
static void load_guard(const double* S, int P, float theta, unsigned char* feas) {
    double tot = 0.0;
    for (int m = 0; m < P; ++m) tot = tot + S[m];
    double Lbar = tot / (double)P;
    double thr = (1.0 + (double)theta) * Lbar;
    for (int m = 0; m < P; ++m) feas[m] = (S[m] <= thr) ? 1 : 0;
}

/* Step 4 of O10 for one token: serve[k] and the accessed set R as a bitmask. */
static uint64_t select_token(const int16_t* T, int k, int home, const int8_t* primary,
                             const int8_t* replicas, int r, const double* S,
                             const unsigned char* feas, int8_t* serve) {
    uint64_t R = 0;
    /* pass 1: forced experts (Q18) */
    for (int j = 0; j < k; ++j) {
        serve[j] = -1;
        int e = T[j];
        if (e < 0) continue;
        int ncand = 1;
        for (int i = 0; i < r; ++i) if (replicas[(size_t)e * r + i] >= 0) ncand++;
        if (ncand == 1) {
            serve[j] = primary[e];
            R |= 1ull << primary[e];
        }
    }
    /* pass 2: replicated experts in slot order; key (non-local, snapshot load, slot) (Q17) */
    for (int j = 0; j < k; ++j) {
        int e = T[j];
        if (e < 0 || serve[j] >= 0) continue;
        int cand[17];
        int nc = 0;
        cand[nc++] = primary[e];
        for (int i = 0; i < r; ++i) if (replicas[(size_t)e * r + i] >= 0) cand[nc++] = replicas[(size_t)e * r + i];
        int anyfeas = 0;
        for (int i = 0; i < nc; ++i) anyfeas |= feas[cand[i]];
        int best = -1, bestloc = 0;
        double bestS = 0.0;
        for (int i = 0; i < nc; ++i) {
            if (anyfeas && !feas[cand[i]]) continue;       /* PAPER.md:155 fallback when none feasible */
            int nonlocal = !(((R >> cand[i]) & 1ull) || cand[i] == home);
            double s = S[cand[i]];
            if (best < 0 || nonlocal < bestloc || (nonlocal == bestloc && s < bestS)) {
                best = i; bestloc = nonlocal; bestS = s;
            }
        }
        serve[j] = (int8_t)cand[best];
        R |= 1ull << cand[best];
    }
    return R;
}

static int popc64(uint64_t x) { int n = 0; while (x) { x &= x - 1; ++n; } return n; }

/* O11 -- fairness.  PAPER.md:453-463 (Eq. 17-18), CV per Q24. */
static void fairness(const uint64_t* load, int P, double* out3) {
    double tot = 0.0, sq = 0.0, mxl = 0.0;
    for (int m = 0; m < P; ++m) {
        double x = (double)load[m];
        tot += x; sq += x * x; if (x > mxl) mxl = x;
    }
    if (tot == 0.0) { out3[0] = 1.0; out3[1] = 0.0; out3[2] = 0.0; return; }
    double mean = tot / P;
    double var = 0.0;
    for (int m = 0; m < P; ++m) { double x = (double)load[m]; var += (x - mean) * (x - mean); }
    var /= P;
    out3[0] = (tot * tot) / (P * sq);
    out3[1] = (mxl - mean) / mean;
    out3[2] = sqrt(var) / mean;
}

/* gesr_select: step 4's serve for one given snapshot.  serve[L,N,k]. */
int orc_gesr_select(const int16_t* indices, int64_t N, int k, int L, int E, int P,
                    const int8_t* primary, const int8_t* replicas, int r,
                    const double* load_snapshot, float theta, int64_t token_offset, int8_t* serve) {
    int use_rep = (replicas != NULL && r > 0);
#pragma omp parallel for schedule(dynamic, 1)
    for (int l = 0; l < L; ++l) {
        unsigned char feas[64];
        const double* S = load_snapshot + (size_t)l * P;
        load_guard(S, P, theta, feas);
        for (int64_t t = 0; t < N; ++t) {
            int home = (int)((token_offset + t) % P);
            select_token(indices + ((size_t)l * N + t) * k, k, home, primary + (size_t)l * E,
                         use_rep ? replicas + (size_t)l * E * r : NULL, use_rep ? r : 0,
                         S, feas, serve + ((size_t)l * N + t) * k);
        }
    }
    return 0;
}

/* O10 + O11.  load[L,P], comm_span[L,F], comm_remote[L,F], ntok[F] are overwritten;
 * load_state[L,P] in/out (NULL: start from 0, discard); fairness[(L+1)*3] fp64;
 * cost_per_token[L,N] and serve[L,N,k] optional. */
int orc_eval(const int16_t* indices, const int8_t* family, int64_t N, int k, int L, int E, int F, int P,
             const int8_t* primary, const int8_t* replicas, int r, float theta, double rho,
             int64_t microbatch, int64_t token_offset, double* load_state, uint64_t* load,
             uint64_t* comm_span, uint64_t* comm_remote, uint64_t* ntok, double* fair,
             uint8_t* cost_per_token, int8_t* serve_out) {
    int use_rep = (replicas != NULL && r > 0);
    int64_t B = (!use_rep || microbatch <= 0) ? N : microbatch;
    memset(load, 0, sizeof(uint64_t) * (size_t)L * P);
    memset(comm_span, 0, sizeof(uint64_t) * (size_t)L * F);
    memset(comm_remote, 0, sizeof(uint64_t) * (size_t)L * F);
    memset(ntok, 0, sizeof(uint64_t) * (size_t)F);
    for (int64_t t = 0; t < N; ++t) {
        int f = family[t];
        if (f >= 0 && f < F) ntok[f] += 1;
    }
#pragma omp parallel for schedule(dynamic, 1)
    for (int l = 0; l < L; ++l) {
        double Ls[64], S[64];
        unsigned char feas[64];
        uint64_t delta[64];
        int8_t sv[16];
        for (int m = 0; m < P; ++m) Ls[m] = load_state ? load_state[(size_t)l * P + m] : 0.0;
        for (int64_t t0 = 0; t0 < N; t0 += B) {
            int64_t t1 = t0 + B < N ? t0 + B : N;
            for (int m = 0; m < P; ++m) { S[m] = Ls[m]; delta[m] = 0; }
            load_guard(S, P, theta, feas);
            for (int64_t t = t0; t < t1; ++t) {
                int f = family[t];
                if (f < 0 || f >= F) {
                    if (serve_out) for (int j = 0; j < k; ++j) serve_out[((size_t)l * N + t) * k + j] = -1;
                    if (cost_per_token) cost_per_token[(size_t)l * N + t] = 0;
                    continue;
                }
                int home = (int)((token_offset + t) % P);
                uint64_t R = select_token(indices + ((size_t)l * N + t) * k, k, home,
                                          primary + (size_t)l * E,
                                          use_rep ? replicas + (size_t)l * E * r : NULL, use_rep ? r : 0,
                                          S, feas, sv);
                for (int j = 0; j < k; ++j) {
                    if (sv[j] >= 0) delta[sv[j]] += 1;
                    if (serve_out) serve_out[((size_t)l * N + t) * k + j] = sv[j];
                }
                int nR = popc64(R);
                int rem = popc64(R & ~(1ull << home));
                comm_span[(size_t)l * F + f] += (uint64_t)(nR > 1 ? nR - 1 : 0);   /* App. C, Q15 */
                comm_remote[(size_t)l * F + f] += (uint64_t)rem;                   /* Q16 */
                if (cost_per_token) cost_per_token[(size_t)l * N + t] = (uint8_t)rem;
            }
            for (int m = 0; m < P; ++m) {                  /* Eq. 15, once per micro-batch (Q19) */
                double prod = rho * Ls[m];
                Ls[m] = prod + (double)delta[m];
                load[(size_t)l * P + m] += delta[m];
            }
        }
        if (load_state) for (int m = 0; m < P; ++m) load_state[(size_t)l * P + m] = Ls[m];
        fairness(load + (size_t)l * P, P, fair + (size_t)l * 3);
    }
    uint64_t tot[64];
    for (int m = 0; m < P; ++m) {
        tot[m] = 0;
        for (int l = 0; l < L; ++l) tot[m] += load[(size_t)l * P + m];
    }
    fairness(tot, P, fair + (size_t)L * 3);
    return 0;
}

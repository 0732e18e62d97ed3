"""ORACLE (definitional form) -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

A plain, slow, obviously-correct CPU statement of what the TACG/GESR hot path
computes, written from the paper (/root/reference/PAPER.md, cited per function
as PAPER.md:<line>) with the readings Q1..Q28 of SURVEY.md 8(c), restated in
DESIGN.md "Readings".  float64 and Python integers throughout, pure-Python
loops, no blocking, fusion or reordering beyond what the text states.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this package.  It shares no code with, and never
imports, paper_2606_01007_b200 (the CUDA path).

Parity pins (tests/test_oracle_pins.py): hand-worked trace of SURVEY.md 8(c)
(tests/golden/handworked_trace.txt), X^T X by numpy.matmul, brute-force
enumeration of Eq. 9, swap-gain identity by recomputing the objective,
closed-form Comm under uniform routing against the paper's printed Baseline
Comm, Jain/MaxVio closed forms, special cases alpha=0,
F=1, identical families, theta=inf, rho in {0,1}; for O14 (spectral-then-repair)
the spectrum of disjoint cliques and of a path, hand-worked repairs, recovery of
planted communities and brute force on tiny graphs.  No function here is
"parity unpinned".
"""
from __future__ import annotations

import itertools
import math
from typing import Dict, Iterator, List, Optional, Sequence, Tuple

import numpy as np


# --------------------------------------------------------------------------
# O1 -- counts (S1, S2).  PAPER.md:71: usage vector u (dispatch frequency of
# each expert) and coactivation matrix A (frequency of expert pairs selected
# by the same token), per layer and family.
# --------------------------------------------------------------------------
def coact_counts(indices: np.ndarray, family: np.ndarray, E: int, F: int):
    """D[l,f,e] dispatch counts, C[l,f,i,j] pair counts (symmetric, zero diagonal),
    ntok[f] tokens per family.  Negative expert id = empty slot, negative family
    = padding token (both skipped; SURVEY.md 8(b) preconditions)."""
    indices = np.asarray(indices)
    family = np.asarray(family)
    L, N, k = indices.shape
    D = np.zeros((L, F, E), dtype=np.int64)
    C = np.zeros((L, F, E, E), dtype=np.int64)
    ntok = np.zeros(F, dtype=np.int64)
    for t in range(N):
        f = int(family[t])
        if f >= 0:
            ntok[f] += 1
    for l in range(L):
        for t in range(N):
            f = int(family[t])
            if f < 0:
                continue
            T = [int(e) for e in indices[l, t] if int(e) >= 0]
            for e in T:
                D[l, f, e] += 1
            for i, j in itertools.combinations(T, 2):
                if i != j:                   # C[l,f,e,e] is never touched
                    C[l, f, i, j] += 1
                    C[l, f, j, i] += 1
    return D, C, ntok


# --------------------------------------------------------------------------
# O2..O5 -- preference scoring.  PAPER.md:71-95 (Eq. 2-6).
# --------------------------------------------------------------------------
def zscore(x: np.ndarray, eps: float) -> np.ndarray:
    """Eq. 4: (x - mu)/(sigma + eps) over experts; population sigma (Q6)."""
    E = len(x)
    mu = sum(float(v) for v in x) / E
    var = sum((float(v) - mu) ** 2 for v in x) / E
    sigma = math.sqrt(var)
    return np.array([(float(v) - mu) / (sigma + eps) for v in x], dtype=np.float64)


def preferences(D: np.ndarray, C: np.ndarray, ntok: np.ndarray, tau: float = 1.0,
                eps: float = 1e-6) -> Dict[str, np.ndarray]:
    """One layer.  D[F,E], C[F,E,E], ntok[F] -> u, c, du, dc, zu, zc, s, pref[E,F]."""
    F, E = D.shape
    u = np.zeros((F, E))
    A = np.zeros((F, E, E))
    c = np.zeros((F, E))
    for f in range(F):
        tot = int(D[f].sum())
        nf = int(ntok[f])
        for e in range(E):
            u[f, e] = float(D[f, e]) / max(1, tot)                 # Q1: relative dispatch frequency
            for e2 in range(E):
                A[f, e, e2] = float(C[f, e, e2]) / max(1, nf)      # Q2: pairs per token of family f
        for e in range(E):
            c[f, e] = sum(abs(A[f, e, e2]) for e2 in range(E))     # Eq. 2 right
    du = np.zeros((F, E))
    dc = np.zeros((F, E))
    for f in range(F):
        for e in range(E):
            if F > 1:                                              # Eq. 2 left, Eq. 3; Q5: F=1 -> 0
                ou = sum(u[g, e] for g in range(F) if g != f) / (F - 1)
                oc = sum(c[g, e] for g in range(F) if g != f) / (F - 1)
            else:
                ou = 0.0
                oc = 0.0
            du[f, e] = u[f, e] - ou
            dc[f, e] = c[f, e] - oc
    zu = np.stack([zscore(du[f], eps) for f in range(F)])
    zc = np.stack([zscore(dc[f], eps) for f in range(F)])
    s = zu + zc                                                    # Eq. 5
    pref = np.zeros((E, F))
    for e in range(E):                                             # Eq. 6, max subtracted
        m = max(s[f, e] / tau for f in range(F))
        ex = [math.exp(s[f, e] / tau - m) for f in range(F)]
        tot = sum(ex)
        for f in range(F):
            pref[e, f] = ex[f] / tot
    return dict(u=u, A=A, c=c, du=du, dc=dc, zu=zu, zc=zc, s=s, pref=pref)


# --------------------------------------------------------------------------
# O6 -- task-modulated graph.  PAPER.md:97-108 (Eq. 7-8).
# --------------------------------------------------------------------------
def graph(C: np.ndarray, ntok: np.ndarray, pref: np.ndarray, alpha: float = 0.25):
    """One layer.  Returns Abar, Ahat, Atask, W (W is the paper's A-tilde)."""
    F, E, _ = C.shape
    Abar = np.zeros((E, E))
    for i in range(E):
        for j in range(E):
            Abar[i, j] = sum(float(C[f, i, j]) / max(1, int(ntok[f])) for f in range(F)) / F
    mx = float(Abar.max()) if E > 0 else 0.0
    Ahat = Abar / mx if mx > 0 else np.zeros_like(Abar)            # Q8
    Atask = np.zeros((E, E))
    for i in range(E):
        for j in range(E):
            Atask[i, j] = sum(pref[i, f] * pref[j, f] for f in range(F))   # Eq. 7
    W = (1.0 - alpha) * Ahat + alpha * (Atask * Ahat)              # Eq. 8
    return Abar, Ahat, Atask, W


# --------------------------------------------------------------------------
# O7, O8 -- affinity (Eq. 10 inner sum) and swap gains
# ("only if the move improves the sum of within-group affinities",
# generalised to all pairs per BASELINE.json north_star).
# --------------------------------------------------------------------------
def affinity(W: np.ndarray, primary: Sequence[int], P: int) -> np.ndarray:
    E = W.shape[0]
    aff = np.zeros((E, P))
    for e in range(E):
        for e2 in range(E):
            aff[e, int(primary[e2])] += W[e, e2]
    return aff


def objective_half(W: np.ndarray, primary: Sequence[int]) -> float:
    """J_half = sum_m sum_{i<j in S_m} W[i,j]: half of Eq. 9's double sum."""
    E = W.shape[0]
    tot = 0.0
    for i in range(E):
        for j in range(i + 1, E):
            if int(primary[i]) == int(primary[j]):
                tot += W[i, j]
    return tot


def swap_gains(W: np.ndarray, aff: np.ndarray, primary: Sequence[int]) -> np.ndarray:
    """G[i,j] = J_half(after exchanging the partitions of i and j) - J_half(before)."""
    E = W.shape[0]
    G = np.zeros((E, E))
    for i in range(E):
        for j in range(E):
            a, b = int(primary[i]), int(primary[j])
            if a != b:
                G[i, j] = aff[i, b] + aff[j, a] - aff[i, a] - aff[j, b] - 2.0 * W[i, j]
    return G


# --------------------------------------------------------------------------
# O9 -- brute force over capacity-feasible placements (Eq. 9).
# --------------------------------------------------------------------------
def enumerate_placements(E: int, P: int, cap: int, labelled: bool = False) -> Iterator[Tuple[int, ...]]:
    """All maps e -> partition with exactly... at most `cap` experts per partition.
    Unlabelled: partitions are interchangeable, a canonical representative is yielded
    (a new partition id may be opened only as the smallest unused one)."""
    assign = [0] * E
    count = [0] * P

    def rec(e: int, used: int):
        if e == E:
            yield tuple(assign)
            return
        limit = P if labelled else min(P, used + 1)
        for m in range(limit):
            if count[m] < cap:
                assign[e] = m
                count[m] += 1
                yield from rec(e + 1, max(used, m + 1))
                count[m] -= 1

    yield from rec(0, 0)


def brute_force_optimum(W: np.ndarray, P: int, cap: int):
    best = -math.inf
    argbest: List[Tuple[int, ...]] = []
    n = 0
    for pl in enumerate_placements(W.shape[0], P, cap, labelled=False):
        n += 1
        j = objective_half(W, pl)
        if j > best + 1e-15:
            best, argbest = j, [pl]
        elif abs(j - best) <= 1e-15:
            argbest.append(pl)
    return best, argbest, n


# --------------------------------------------------------------------------
# O10 -- GESR serving selection + evaluation (S8-S11).
# PAPER.md:145-159 (Eq. 13-15), Comm per PAPER.md:363 (App. C), readings Q15-Q23.
# --------------------------------------------------------------------------
def load_guard(S: Sequence[float], theta: float) -> List[bool]:
    """Eq. 13-14: feas[m] = S[m] <= (1+theta) * mean(S); mean summed left to right."""
    P = len(S)
    tot = 0.0
    for m in range(P):
        tot = tot + float(S[m])
    Lbar = tot / P
    thr = (1.0 + float(np.float32(theta))) * Lbar          # theta is a float widened to double (Q19)
    return [float(S[m]) <= thr for m in range(P)]


def select_token(experts: Sequence[int], home: int, primary: Sequence[int],
                 replicas: Optional[np.ndarray], S: Sequence[float], feas: Sequence[bool]):
    """Step 4 of O10 for one token of one layer.  Returns serve[k] (-1 for empty slots) and R."""
    k = len(experts)
    serve = [-1] * k
    R = set()

    def cand(e):
        c = [int(primary[e])]
        if replicas is not None:
            c += [int(x) for x in replicas[e] if int(x) >= 0]
        return c

    # Pass 1: forced experts (single candidate) are accessed regardless (Q18).
    for j in range(k):
        e = int(experts[j])
        if e < 0:
            continue
        c = cand(e)
        if len(c) == 1:
            serve[j] = c[0]
            R.add(c[0])
    # Pass 2: replicated experts in slot order; locality, then snapshot load, then slot (Q17).
    for j in range(k):
        e = int(experts[j])
        if e < 0:
            continue
        c = cand(e)
        if len(c) == 1:
            continue
        Fs = [i for i in range(len(c)) if feas[c[i]]]
        if not Fs:
            Fs = list(range(len(c)))                       # PAPER.md:155 fallback
        best = min(Fs, key=lambda i: (0 if (c[i] in R or c[i] == home) else 1, float(S[c[i]]), i))
        serve[j] = c[best]
        R.add(c[best])
    return serve, R


def eval_placement(indices: np.ndarray, family: np.ndarray, E: int, F: int, P: int,
                   primary: np.ndarray, replicas: Optional[np.ndarray] = None,
                   theta: float = 0.15, rho: float = 0.995, microbatch: int = 0,
                   load_state: Optional[np.ndarray] = None, token_offset: int = 0):
    """All layers.  Returns dict(load[L,P], comm_span[L,F], comm_remote[L,F], ntok[F],
    fairness[L+1,3], cost[L,N], serve[L,N,k], load_state[L,P])."""
    indices = np.asarray(indices)
    family = np.asarray(family)
    L, N, k = indices.shape
    r = 0 if replicas is None else replicas.shape[2]
    use_rep = replicas is not None and r > 0
    B = N if (not use_rep or microbatch <= 0) else int(microbatch)
    load = np.zeros((L, P), dtype=np.int64)
    span = np.zeros((L, F), dtype=np.int64)
    remote = np.zeros((L, F), dtype=np.int64)
    cost = np.zeros((L, N), dtype=np.int64)
    serve_all = np.full((L, N, k), -1, dtype=np.int64)
    ntok = np.zeros(F, dtype=np.int64)
    for t in range(N):
        if int(family[t]) >= 0:
            ntok[int(family[t])] += 1
    state = np.zeros((L, P), dtype=np.float64) if load_state is None else np.array(load_state, dtype=np.float64)
    for l in range(L):
        Ls = [float(x) for x in state[l]]
        t0 = 0
        while t0 < N:
            t1 = min(N, t0 + B)
            S = list(Ls)                                    # step 1: snapshot
            feas = load_guard(S, theta)                     # steps 2-3
            delta = [0] * P
            for t in range(t0, t1):                         # step 4
                f = int(family[t])
                if f < 0:
                    continue
                home = (token_offset + t) % P
                sv, R = select_token(indices[l, t], home, primary[l],
                                     replicas[l] if use_rep else None, S, feas)
                for j in range(k):
                    if sv[j] >= 0:
                        delta[sv[j]] += 1
                        serve_all[l, t, j] = sv[j]
                span[l, f] += max(0, len(R) - 1)            # Comm, App. C (Q15)
                rem = len(R - {home})                       # remote-partition cost (Q16)
                remote[l, f] += rem
                cost[l, t] = rem
            for m in range(P):                              # step 5: Eq. 15 once per micro-batch (Q19)
                prod = float(np.float64(rho) * np.float64(Ls[m]))     # one rounded multiply
                Ls[m] = float(np.float64(prod) + np.float64(delta[m]))  # one rounded add
                load[l, m] += delta[m]
            t0 = t1
        state[l] = Ls
    fair = np.zeros((L + 1, 3), dtype=np.float64)
    for l in range(L):
        fair[l] = fairness(load[l])
    fair[L] = fairness(load.sum(axis=0))
    return dict(load=load, comm_span=span, comm_remote=remote, ntok=ntok, fairness=fair,
                cost=cost, serve=serve_all, load_state=state)


def gesr_select(indices: np.ndarray, E: int, P: int, primary: np.ndarray,
                replicas: Optional[np.ndarray], load_snapshot: np.ndarray, theta: float,
                token_offset: int = 0) -> np.ndarray:
    """serve[L,N,k] for one given snapshot (step 4 of O10 only)."""
    L, N, k = indices.shape
    out = np.full((L, N, k), -1, dtype=np.int64)
    use_rep = replicas is not None and replicas.shape[2] > 0
    for l in range(L):
        S = [float(x) for x in load_snapshot[l]]
        feas = load_guard(S, theta)
        for t in range(N):
            home = (token_offset + t) % P
            sv, _ = select_token(indices[l, t], home, primary[l],
                                 replicas[l] if use_rep else None, S, feas)
            out[l, t] = sv
    return out


# --------------------------------------------------------------------------
# O11 -- fairness (S12).  PAPER.md:453-463 (Eq. 17-18); CV per Q24.
# --------------------------------------------------------------------------
def fairness(load: Sequence[int]) -> Tuple[float, float, float]:
    P = len(load)
    Ls = [float(x) for x in load]
    tot = sum(Ls)
    if tot == 0.0:
        return (1.0, 0.0, 0.0)
    sq = sum(x * x for x in Ls)
    mean = tot / P
    jain = (tot * tot) / (P * sq)
    maxvio = (max(Ls) - mean) / mean
    var = sum((x - mean) ** 2 for x in Ls) / P
    cv = math.sqrt(var) / mean
    return (jain, maxvio, cv)


# --------------------------------------------------------------------------
# O12 -- harness helpers (make inputs; not graded as kernels).
# --------------------------------------------------------------------------
def default_placement(E: int, capacity: int) -> np.ndarray:
    return np.array([e // capacity for e in range(E)], dtype=np.int64)


def local_search(W: np.ndarray, P: int, capacity: int, max_swaps: Optional[int] = None):
    """Capacity-preserving best-swap local search standing in for the consumers of
    PAPER.md:119-124 (not the paper's spectral method).  Returns (primary, n_swaps)."""
    E = W.shape[0]
    primary = default_placement(E, capacity)
    if max_swaps is None:
        max_swaps = 4 * E
    n = 0
    while n < max_swaps:
        aff = affinity(W, primary, P)
        G = swap_gains(W, aff, primary)
        bi, bj, bg = -1, -1, 0.0
        for i in range(E):
            for j in range(i + 1, E):
                if G[i, j] > bg:
                    bi, bj, bg = i, j, G[i, j]
        if bi < 0:
            break
        a, b = int(primary[bi]), int(primary[bj])
        terms = abs(aff[bi, b]) + abs(aff[bj, a]) + abs(aff[bi, a]) + abs(aff[bj, b]) + 2 * abs(W[bi, bj])
        if not bg > 1e-7 * terms:
            break
        primary[bi], primary[bj] = b, a
        n += 1
    return primary, n


def replica_table(Abar: np.ndarray, aff: np.ndarray, primary: Sequence[int], n_rep: int, r: int) -> np.ndarray:
    """Generic experts = top n_rep by Cent_e = sum_e' Abar[e,e'] (Eq. 11 with
    lambda1=lambda2=0); secondaries = r non-primary partitions
    with largest aff.  Ties -> lower id."""
    E, P = aff.shape
    cent = [float(sum(Abar[e])) for e in range(E)]
    order = sorted(range(E), key=lambda e: (-cent[e], e))
    rep = np.full((E, r), -1, dtype=np.int64)
    for e in order[:n_rep]:
        cands = sorted((m for m in range(P) if m != int(primary[e])), key=lambda m: (-aff[e, m], m))
        for i, m in enumerate(cands[:r]):
            rep[e, i] = m
    return rep


# --------------------------------------------------------------------------
# O13 -- GESR offline scoring with lambda1, lambda2 != 0.
# PAPER.md:132-138, Eq. 11: r_e = Cent_e + lambda1 Cons_e - lambda2 Spec_e with
#   Cent_e = sum_e' Abar[e,e']                                   (pooled coactivation)
#   Cons_e = average over families of the cosine similarity between the expert's
#            family-specific coactivation profile A^f[e,:] and the mean profile Abar[e,:]
#   Spec_e = maximum deviation from that mean profile across families.
# Readings (Q29-Q31): the cosine of a zero vector with anything is 0; the
# "deviation" is the Euclidean norm of A^f[e,:] - Abar[e,:]; ties in the top-n_rep
# selection and among secondaries go to the lower id.  A^f and Abar as in O2/O6
# (A^f = C^f / max(1, N_f), Abar = mean over families, readings Q2, Q4).
# --------------------------------------------------------------------------
def gesr_scores(C: np.ndarray, ntok: np.ndarray, lam1: float, lam2: float) -> Dict[str, np.ndarray]:
    """C: counts [F,E,E] of one layer; returns cent, cons, spec, score as float64[E]."""
    F, E, _ = C.shape
    A = [[[float(C[f][i][j]) / max(1.0, float(ntok[f])) for j in range(E)] for i in range(E)] for f in range(F)]
    Abar = [[sum(A[f][i][j] for f in range(F)) / F for j in range(E)] for i in range(E)]
    cent, cons, spec, score = [], [], [], []
    for e in range(E):
        mean = Abar[e]
        nm = math.sqrt(sum(v * v for v in mean))
        c_e = sum(mean)
        cos_sum = 0.0
        dev_max = 0.0
        for f in range(F):
            row = A[f][e]
            nr = math.sqrt(sum(v * v for v in row))
            dot = sum(row[j] * mean[j] for j in range(E))
            cos_sum += dot / (nr * nm) if nr > 0.0 and nm > 0.0 else 0.0
            dev = math.sqrt(sum((row[j] - mean[j]) ** 2 for j in range(E)))
            dev_max = max(dev_max, dev)
        cent.append(c_e)
        cons.append(cos_sum / F)
        spec.append(dev_max)
        score.append(c_e + lam1 * (cos_sum / F) - lam2 * dev_max)
    return {"cent": np.array(cent), "cons": np.array(cons), "spec": np.array(spec), "score": np.array(score)}


def gesr_replica_table(score: Sequence[float], aff: np.ndarray, primary: Sequence[int], n_rep: int, r: int) -> np.ndarray:
    """Eq. 12: the n_rep top-scoring experts keep their primary and receive the r non-primary
    partitions with the largest affinity aff[e,m]; -1 elsewhere.  Ties -> lower id."""
    E, P = aff.shape
    order = sorted(range(E), key=lambda e: (-float(score[e]), e))
    rep = np.full((E, r), -1, dtype=np.int64)
    for e in order[:n_rep]:
        cands = sorted((m for m in range(P) if m != int(primary[e])), key=lambda m: (-float(aff[e, m]), m))
        for i, m in enumerate(cands[:r]):
            rep[e, i] = m
    return rep


# --------------------------------------------------------------------------
# O14 -- capacity-feasible expert grouping, spectral-then-repair.
# PAPER.md:117-124.  Stage 1: "symmetrize A-tilde, scale it to [0,1], add a small diagonal jitter
# ... form the symmetric normalized Laplacian L_sym = I - D^-1/2 A D^-1/2 with degree matrix D,
# embed experts via its M smallest eigenvectors, and run k-means with k = M".  Stage 2: every
# overfull group keeps its top-C_m members by intra-group affinity, the rest enter an overflow
# pool and are inserted greedily by Eq. 10.
# Readings (Q33-Q37): scale = divide by the largest entry; jitter 1e-6; the degree
# includes the jitter; rows of the embedding are not renormalised (the text does not say so);
# k-means is Lloyd's iteration from a deterministic farthest-point start (first centre = the
# expert of largest degree, then the expert farthest from the chosen centres), an empty cluster
# keeps its centre, ties go to the lower id everywhere; C_m = capacity is an upper bound when
# E < M*capacity; the pool is served group by group, strongest evicted member first.  After the
# greedy pass every expert sits in a group of size <= C_m (a non-full group always exists while
# sum C_m >= E), so the donor-receiver loop of PAPER.md:124 has nothing left to move: it is
# stated here as a check, not as code.
# --------------------------------------------------------------------------
def scaled_affinity(W: np.ndarray) -> np.ndarray:
    """(W + W^T)/2 divided by its largest entry (all zeros stay all zeros).  float64[E,E]."""
    E = W.shape[0]
    S = [[(float(W[i][j]) + float(W[j][i])) * 0.5 for j in range(E)] for i in range(E)]
    top = max(max(row) for row in S)
    if top > 0.0:
        S = [[v / top for v in row] for row in S]
    return np.array(S, dtype=np.float64)


def spectral_embedding(W: np.ndarray, M: int, jitter: float = 1e-6):
    """Returns (X float64[E,M], eigenvalues float64[M]): the eigenvectors of the M smallest
    eigenvalues of L_sym of the scaled, jittered affinity (columns in increasing eigenvalue
    order; an eigenvector's sign, and the basis inside a repeated eigenvalue, are not unique)."""
    S = scaled_affinity(W)
    E = S.shape[0]
    A = S + jitter * np.eye(E)
    deg = A.sum(axis=1)
    inv = 1.0 / np.sqrt(deg)
    Lsym = np.eye(E) - inv[:, None] * A * inv[None, :]
    vals, vecs = np.linalg.eigh(Lsym)            # library step: symmetric eigendecomposition, ascending
    return vecs[:, :M].copy(), vals[:M].copy()


def kmeans_labels(X: np.ndarray, k: int, first: int, iters: int = 100) -> List[int]:
    """Lloyd's k-means on the rows of X from a farthest-point start whose first centre is row `first`."""
    E = X.shape[0]

    def d2(a, b):
        return float(sum((float(a[t]) - float(b[t])) ** 2 for t in range(len(a))))

    centres = [list(map(float, X[first]))]
    mind = [d2(X[e], centres[0]) for e in range(E)]
    while len(centres) < k:
        nxt = max(range(E), key=lambda e: (mind[e], -e))
        centres.append(list(map(float, X[nxt])))
        for e in range(E):
            mind[e] = min(mind[e], d2(X[e], centres[-1]))
    labels = [-1] * E
    for _ in range(iters):
        new = [min(range(k), key=lambda c: (d2(X[e], centres[c]), c)) for e in range(E)]
        if new == labels:
            break
        labels = new
        for c in range(k):
            members = [e for e in range(E) if labels[e] == c]
            if members:
                centres[c] = [sum(float(X[e][t]) for e in members) / len(members) for t in range(X.shape[1])]
    return labels


def capacity_repair(S: np.ndarray, labels0: Sequence[int], P: int, capacity: int) -> List[int]:
    """Stage 2 on the scaled affinity S (self-affinity never counted)."""
    E = S.shape[0]
    groups = [[e for e in range(E) if int(labels0[e]) == m] for m in range(P)]
    pool: List[int] = []
    for m in range(P):
        if len(groups[m]) > capacity:
            intra = {e: sum(float(S[e][e2]) for e2 in groups[m] if e2 != e) for e in groups[m]}
            ranked = sorted(groups[m], key=lambda e: (-intra[e], e))
            groups[m] = sorted(ranked[:capacity])
            pool.extend(ranked[capacity:])
    for e in pool:
        open_groups = [m for m in range(P) if len(groups[m]) < capacity]
        inc = {m: sum(float(S[e][e2]) for e2 in groups[m]) for m in open_groups}       # Eq. 10
        best = max(open_groups, key=lambda m: (inc[m], -m))
        groups[best] = sorted(groups[best] + [e])
    assert all(len(g) <= capacity for g in groups)        # nothing left for the donor-receiver loop
    out = [-1] * E
    for m in range(P):
        for e in groups[m]:
            out[e] = m
    return out


def spectral_place(W: np.ndarray, P: int, capacity: int, jitter: float = 1e-6, iters: int = 100):
    """Stage 1 + Stage 2 for one layer.  Returns (primary list[E], labels0 list[E], X float64[E,P])."""
    E = W.shape[0]
    assert E <= P * capacity
    X, _ = spectral_embedding(W, P, jitter)
    S = scaled_affinity(W)
    deg = [sum(float(S[e][e2]) for e2 in range(E)) + jitter for e in range(E)]
    first = max(range(E), key=lambda e: (deg[e], -e))
    labels0 = kmeans_labels(X, P, first, iters)
    return capacity_repair(S, labels0, P, capacity), labels0, X


# --------------------------------------------------------------------------
# O15 -- motivation diagnostics.  PAPER.md:469: "The activation Frobenius
# distance between two task families is the Frobenius norm ||P_i - P_j||_F of the difference
# between their expert-activation distributions ... The top-64 pair Jaccard overlap measures the
# Jaccard similarity between the sets of top-64 most frequently coactivated expert pairs of two
# task families."
# Readings (Q38): P_f[l,e] = D[l,f,e] / max(1, N_f), the per-expert activation
# probability of the same paragraph; the distance is reported per layer (the 2-norm of a row) and
# over the whole [L,E] matrix (row L of the output); the top pairs are taken per layer among pairs
# that co-activated at least once, most frequent first, ties -> smaller (i,j); the Jaccard
# similarity of two empty sets is 0; row L is the mean over layers.
# --------------------------------------------------------------------------
def top_pairs(Cf: np.ndarray, topk: int = 64) -> List[Tuple[int, int]]:
    """The topk unordered pairs (i<j) of one family's count matrix, most frequent first."""
    E = Cf.shape[0]
    pairs = [(i, j) for i in range(E) for j in range(i + 1, E) if int(Cf[i][j]) > 0]
    pairs.sort(key=lambda ij: (-int(Cf[ij[0]][ij[1]]), ij[0], ij[1]))
    return pairs[:topk]


def family_divergence(D: np.ndarray, C: np.ndarray, ntok: np.ndarray, topk: int = 64):
    """D [L,F,E], C [L,F,E,E], ntok [F] -> (frob float64[L+1,F,F], jaccard float64[L+1,F,F])."""
    L, F, E = D.shape
    frob = np.zeros((L + 1, F, F))
    jac = np.zeros((L + 1, F, F))
    sq_all = [[0.0] * F for _ in range(F)]
    for l in range(L):
        P = [[float(D[l][f][e]) / max(1.0, float(ntok[f])) for e in range(E)] for f in range(F)]
        sets = [set(top_pairs(C[l][f], topk)) for f in range(F)]
        for f in range(F):
            for g in range(F):
                sq = sum((P[f][e] - P[g][e]) ** 2 for e in range(E))
                frob[l, f, g] = math.sqrt(sq)
                sq_all[f][g] += sq
                union = len(sets[f] | sets[g])
                jac[l, f, g] = len(sets[f] & sets[g]) / union if union else 0.0
    for f in range(F):
        for g in range(F):
            frob[L, f, g] = math.sqrt(sq_all[f][g])
            jac[L, f, g] = sum(jac[l, f, g] for l in range(L)) / L
    return frob, jac

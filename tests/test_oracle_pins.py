"""Pins the oracle (oracle/ref.py) to things other than itself: the hand-worked trace,
library routines, brute force, closed forms, invariants and special cases
(SURVEY.md 8(c) "What pins each part").  CPU only."""
import itertools
import math
from collections import Counter

import numpy as np
import pytest

from oracle import ref
from tests.conftest import load_golden
import tracegen


def _arr(rows):
    return np.array(rows, dtype=np.float64)


def _hand(golden_trace):
    g = golden_trace
    E, k, F, P = (int(g[x][0][0]) for x in ("E", "k", "F", "P"))
    fam = np.array(g["family"][0], dtype=np.int64)
    idx = np.array(g["experts"], dtype=np.int64)[None]          # [1,N,k]
    return g, E, k, F, P, fam, idx


# ---------------------------------------------------------------- hand-worked trace
def test_handworked_counts(golden_trace):
    g, E, k, F, P, fam, idx = _hand(golden_trace)
    D, C, ntok = ref.coact_counts(idx, fam, E, F)
    assert D[0, 0].tolist() == g["D0"][0] and D[0, 1].tolist() == g["D1"][0]
    Cexp = np.zeros((F, E, E), dtype=np.int64)
    for f, i, j, c in g["C"]:
        Cexp[int(f), int(i), int(j)] = Cexp[int(f), int(j), int(i)] = int(c)
    assert (C[0] == Cexp).all()
    assert ntok.tolist() == [4, 4]


def test_handworked_preferences_graph(golden_trace):
    g, E, k, F, P, fam, idx = _hand(golden_trace)
    D, C, ntok = ref.coact_counts(idx, fam, E, F)
    pr = ref.preferences(D[0], C[0], ntok, tau=g["tau"][0][0], eps=g["eps"][0][0])
    tol = 1.5e-6
    assert np.allclose(pr["u"], [g["u0"][0], g["u1"][0]], atol=tol)
    assert np.allclose(pr["c"], [g["c0"][0], g["c1"][0]], atol=tol)
    assert np.allclose(pr["du"][0], g["du0"][0], atol=tol) and np.allclose(pr["du"][1], -_arr(g["du0"][0]), atol=tol)
    assert np.allclose(pr["dc"][0], g["dc0"][0], atol=tol)
    assert np.allclose(pr["zu"][0], g["zu0"][0], atol=tol)
    assert np.allclose(pr["zc"][0], g["zc0"][0], atol=tol)
    assert np.allclose(pr["s"][0], g["s0"][0], atol=2 * tol) and np.allclose(pr["s"][1], -_arr(g["s0"][0]), atol=2 * tol)
    assert np.allclose(pr["pref"], _arr(g["pref"]), atol=tol)
    Abar, Ahat, Atask, W = ref.graph(C[0], ntok, pr["pref"], alpha=g["alpha"][0][0])
    assert np.allclose(Abar, _arr(g["Abar"]), atol=tol)
    assert np.allclose(Ahat, _arr(g["Ahat"]), atol=tol)
    assert np.allclose(W, _arr(g["W"]), atol=tol)
    # objective of the three unlabelled placements, optimum {01|23}
    J = [ref.objective_half(W, p) for p in ([0, 0, 1, 1], [0, 1, 0, 1], [0, 1, 1, 0])]
    assert np.allclose(J, g["J"][0], atol=2 * tol)
    best, arg, n = ref.brute_force_optimum(W, P, 2)
    assert n == 3 and arg == [(0, 0, 1, 1)] and abs(best - g["J"][0][0]) < 2 * tol
    primary = [int(x) for x in g["primary"][0]]
    aff = ref.affinity(W, primary, P)
    assert np.allclose(aff, _arr(g["aff"]), atol=tol)
    G = ref.swap_gains(W, aff, primary)
    Gexp = np.zeros((E, E))
    for i, j, v in g["G"]:
        Gexp[int(i), int(j)] = Gexp[int(j), int(i)] = v
    assert np.allclose(G, Gexp, atol=3 * tol)


def test_handworked_eval_no_replicas(golden_trace):
    g, E, k, F, P, fam, idx = _hand(golden_trace)
    primary = np.array(g["primary"], dtype=np.int64)
    out = ref.eval_placement(idx, fam, E, F, P, primary)
    assert out["load"][0].tolist() == g["load"][0]
    assert out["comm_span"][0].tolist() == g["comm_span"][0]
    assert out["comm_remote"][0].tolist() == g["comm_remote"][0]
    j, mv, cv = out["fairness"][0]
    assert abs(j - g["jain"][0][0]) < 1.5e-6 and abs(mv - g["maxvio"][0][0]) < 1e-12 and abs(cv - g["cv"][0][0]) < 1e-12
    assert (out["serve"][0] == primary[0][idx[0]]).all()


def test_handworked_eval_gesr(golden_trace):
    g, E, k, F, P, fam, idx = _hand(golden_trace)
    primary = np.array(g["primary"], dtype=np.int64)
    replicas = np.array(g["gesr_replicas"], dtype=np.int64)[None]          # [1,E,1]
    B = int(g["gesr_B"][0][0])
    th, rho = g["theta"][0][0], g["rho"][0][0]
    out = ref.eval_placement(idx, fam, E, F, P, primary, replicas, theta=th, rho=rho, microbatch=B)
    assert out["serve"][0].tolist() == [[int(x) for x in r] for r in g["gesr_serve"]]
    assert out["load"][0].tolist() == g["gesr_load"][0]
    assert int(out["comm_span"].sum()) == g["gesr_comm_span_total"][0][0]
    assert int(out["comm_remote"].sum()) == g["gesr_comm_remote_total"][0][0]
    assert np.allclose(out["load_state"][0], g["gesr_state_final"][0], rtol=0, atol=1e-12)
    assert abs(out["fairness"][0][0] - g["gesr_jain"][0][0]) < 1.5e-6
    assert abs(out["fairness"][0][1] - g["gesr_maxvio"][0][0]) < 1e-12
    # first micro-batch alone
    out0 = ref.eval_placement(idx[:, :B], fam[:B], E, F, P, primary, replicas, theta=th, rho=rho, microbatch=B)
    assert out0["load_state"][0].tolist() == g["gesr_state_mb0"][0]
    # gesr_select with the snapshot of micro-batch 1 reproduces its serve rows
    sv = ref.gesr_select(idx[:, B:], E, P, primary, replicas, np.array([g["gesr_state_mb0"][0]]), th, token_offset=B)
    assert sv[0].tolist() == [[int(x) for x in r] for r in g["gesr_serve"][B:]]


# ---------------------------------------------------------------- counts (O1)
def _small_trace(seed=3, E=12, k=3, L=2, F=3, N=300):
    cfg = tracegen.TraceConfig(name="t", E=E, k=k, L=L, F=F, N=N, N_eval=N, P=4, capacity=3,
                               mix=tuple([1.0 / F] * F), mix_eval=tuple([1.0 / F] * F),
                               popularity="dirichlet", pop_param=0.5, group_size=3, p_group=0.6,
                               n_generic=0, generic_mass=0, generic_mass_eval=0, r=0, n_rep=0,
                               microbatch=64, seed=seed)
    idx, fam = tracegen.gen_trace(cfg)
    return cfg, idx.numpy(), fam.numpy()


def test_counts_matmul_and_invariants():
    cfg, idx, fam = _small_trace()
    E, F, k = cfg.E, cfg.F, cfg.k
    D, C, ntok = ref.coact_counts(idx, fam, E, F)
    L, N, _ = idx.shape
    for l in range(L):
        for f in range(F):
            X = np.zeros((N, E), dtype=np.int64)
            for t in range(N):
                if fam[t] == f:
                    X[t, idx[l, t]] = 1
            G = X.T @ X                                    # library routine: Gram matrix
            assert (np.diag(G) == D[l, f]).all()
            off = G - np.diag(np.diag(G))
            assert (off == C[l, f]).all()
            assert (C[l, f] == C[l, f].T).all() and (np.diag(C[l, f]) == 0).all()
            assert D[l, f].sum() == k * ntok[f]
        assert sum(np.triu(C[l, f], 1).sum() for f in range(F)) == N * k * (k - 1) // 2
    assert ntok.sum() == N


def test_counts_bruteforce_counter_additive_permutation():
    cfg, idx, fam = _small_trace(seed=5, N=200)
    E, F = cfg.E, cfg.F
    D, C, ntok = ref.coact_counts(idx, fam, E, F)
    cnt = Counter()
    for l in range(idx.shape[0]):
        for t in range(idx.shape[1]):
            for i, j in itertools.combinations(sorted(idx[l, t].tolist()), 2):
                cnt[(l, int(fam[t]), i, j)] += 1
    for (l, f, i, j), v in cnt.items():
        assert C[l, f, i, j] == v == C[l, f, j, i]
    assert sum(cnt.values()) == np.triu(C.sum(axis=1), 1).sum()
    # additivity: two halves add up to the whole
    h = 77
    D1, C1, n1 = ref.coact_counts(idx[:, :h], fam[:h], E, F)
    D2, C2, n2 = ref.coact_counts(idx[:, h:], fam[h:], E, F)
    assert (D1 + D2 == D).all() and (C1 + C2 == C).all() and (n1 + n2 == ntok).all()
    # permuting tokens changes nothing
    perm = np.random.default_rng(0).permutation(idx.shape[1])
    Dp, Cp, _ = ref.coact_counts(idx[:, perm], fam[perm], E, F)
    assert (Dp == D).all() and (Cp == C).all()


def test_counts_empty_slots_and_padding():
    idx = np.array([[[0, 1, -1], [2, -1, 3], [1, 2, 0]]])
    fam = np.array([0, -1, 1])
    D, C, ntok = ref.coact_counts(idx, fam, 4, 2)
    assert D[0, 0].tolist() == [1, 1, 0, 0] and D[0, 1].tolist() == [1, 1, 1, 0]
    assert C[0, 0, 0, 1] == 1 and C[0, 0].sum() == 2 and C[0, 1].sum() == 6
    assert ntok.tolist() == [1, 1]


# ---------------------------------------------------------------- preferences / graph (O2-O6)
def _stats(seed=7, **kw):
    cfg, idx, fam = _small_trace(seed=seed, **kw)
    D, C, ntok = ref.coact_counts(idx, fam, cfg.E, cfg.F)
    return cfg, D, C, ntok


def test_pref_rows_sum_to_one_and_relabel():
    cfg, D, C, ntok = _stats()
    pr = ref.preferences(D[0], C[0], ntok)
    assert np.allclose(pr["pref"].sum(axis=1), 1.0, atol=1e-14)
    perm = [2, 0, 1]
    pr2 = ref.preferences(D[0][perm], C[0][perm], ntok[perm])
    assert np.allclose(pr2["pref"], pr["pref"][:, perm], atol=1e-12)


def test_pref_special_cases():
    cfg, D, C, ntok = _stats(F=1, seed=9)
    pr = ref.preferences(D[0], C[0], ntok)
    assert (pr["pref"] == 1.0).all()                                  # F=1 -> pref == 1 (Q5)
    Abar, Ahat, Atask, W = ref.graph(C[0], ntok, pr["pref"], alpha=0.7)
    assert np.allclose(W, Ahat, atol=1e-15)                           # F=1 -> W = Ahat for every alpha
    # identical families -> Delta = 0 -> pref = 1/F exactly
    cfg, D, C, ntok = _stats(F=3, seed=11)
    D2 = np.stack([D[0, 0]] * 3)
    C2 = np.stack([C[0, 0]] * 3)
    n2 = np.array([ntok[0]] * 3)
    pr = ref.preferences(D2, C2, n2)
    assert (pr["pref"] == 1.0 / 3).all()
    Abar, Ahat, Atask, W = ref.graph(C2, n2, pr["pref"], alpha=0.25)
    assert np.allclose(W, Ahat * (1 - 0.25 + 0.25 / 3), atol=1e-15)   # pref == 1/F -> W = Ahat(1-a+a/F)
    # tau -> large -> pref -> 1/F
    cfg, D, C, ntok = _stats(F=3, seed=13)
    pr = ref.preferences(D[0], C[0], ntok, tau=1e9)
    assert np.allclose(pr["pref"], 1.0 / 3, atol=1e-7)


def test_zscore_against_numpy():
    x = np.random.default_rng(1).normal(size=37)
    z = ref.zscore(x, 1e-6)
    assert np.allclose(z, (x - x.mean()) / (x.std() + 1e-6), atol=1e-13)     # numpy std is population std


def test_graph_invariants():
    cfg, D, C, ntok = _stats(seed=17, E=16, N=500)
    pr = ref.preferences(D[0], C[0], ntok)
    for alpha in (0.0, 0.25, 1.0):
        Abar, Ahat, Atask, W = ref.graph(C[0], ntok, pr["pref"], alpha=alpha)
        assert np.allclose(W, W.T, atol=1e-15) and (np.diag(W) == 0).all()
        assert W.min() >= 0 and W.max() <= 1 + 1e-15 and abs(Ahat.max() - 1.0) < 1e-15
        assert ((W == 0) == (Abar == 0)).all() or alpha == 1.0      # no new edges
        assert (W[Abar == 0] == 0).all()
        assert (W <= Ahat + 1e-15).all() and (W >= (1 - alpha) * Ahat - 1e-15).all()
        if alpha == 0.0:
            assert np.allclose(W, Ahat, atol=1e-15)                  # alpha=0: task-agnostic
        # Abar is the library mean of the per-family rates
        assert np.allclose(Abar, np.mean([C[0][f] / max(1, ntok[f]) for f in range(cfg.F)], axis=0), atol=1e-15)
        assert np.allclose(Atask, pr["pref"] @ pr["pref"].T, atol=1e-15)      # Eq. 7 by numpy.matmul


# ---------------------------------------------------------------- affinity / gains / Eq. 9 (O7-O9)
def test_affinity_and_gain_identity():
    cfg, D, C, ntok = _stats(seed=19, E=12, N=400)
    E, P, cap = 12, 4, 3
    pr = ref.preferences(D[0], C[0], ntok)
    _, _, _, W = ref.graph(C[0], ntok, pr["pref"])
    primary = tracegen.random_placement(E, P, cap, 1, seed=4)[0].astype(np.int64)
    aff = ref.affinity(W, primary, P)
    M = np.zeros((E, P))
    M[np.arange(E), primary] = 1
    assert np.allclose(aff, W @ M, atol=1e-14)                                  # numpy.matmul
    assert np.allclose(aff.sum(axis=1), W.sum(axis=1), atol=1e-13)
    J = ref.objective_half(W, primary)
    assert abs(sum(aff[e, primary[e]] for e in range(E)) - 2 * J) < 1e-12
    G = ref.swap_gains(W, aff, primary)
    assert np.allclose(G, G.T, atol=1e-13)
    for i in range(E):
        for j in range(E):
            if primary[i] == primary[j]:
                assert G[i, j] == 0.0
            else:
                p2 = primary.copy()
                p2[i], p2[j] = primary[j], primary[i]
                assert abs(G[i, j] - (ref.objective_half(W, p2) - J)) < 1e-12      # recomputed from scratch


def test_enumeration_counts():
    assert sum(1 for _ in ref.enumerate_placements(8, 4, 2)) == 105               # 8!/((2!)^4 4!)
    assert sum(1 for _ in ref.enumerate_placements(8, 4, 2, labelled=True)) == 2520
    assert sum(1 for _ in ref.enumerate_placements(6, 2, 3)) == 10                # C(6,3)/2
    for pl in ref.enumerate_placements(6, 3, 2, labelled=True):
        assert max(Counter(pl).values()) <= 2


def test_tiny_bruteforce_matching_and_local_search():
    cfg = tracegen.get_config(1)
    idx, fam = tracegen.gen_trace(cfg)
    idx, fam = idx.numpy(), fam.numpy()
    D, C, ntok = ref.coact_counts(idx, fam, cfg.E, cfg.F)
    pr = ref.preferences(D[0], C[0], ntok)
    _, _, _, W = ref.graph(C[0], ntok, pr["pref"])
    best, arg, n = ref.brute_force_optimum(W, cfg.P, cfg.capacity)
    assert n == 105
    # cap = 2: Eq. 9 is maximum-weight perfect matching; independent enumeration of perfect matchings
    def matchings(items):
        if not items:
            yield []
            return
        a = items[0]
        for i in range(1, len(items)):
            rest = items[1:i] + items[i + 1:]
            for m in matchings(rest):
                yield [(a, items[i])] + m
    mbest = max(sum(W[a, b] for a, b in m) for m in matchings(list(range(cfg.E))))
    assert abs(best - mbest) < 1e-12
    try:
        from scipy.sparse.csgraph import min_weight_full_bipartite_matching  # noqa: F401
    except Exception:
        pass
    primary, nsw = ref.local_search(W, cfg.P, cfg.capacity)
    assert max(Counter(primary.tolist()).values()) <= cfg.capacity
    aff = ref.affinity(W, primary, cfg.P)
    G = ref.swap_gains(W, aff, primary)
    assert G.max() <= 1e-6                                        # local optimum: no positive gain
    J = ref.objective_half(W, primary)
    assert J <= best + 1e-12 and J >= ref.objective_half(W, ref.default_placement(cfg.E, cfg.capacity)) - 1e-12


# ---------------------------------------------------------------- evaluation (O10)
def test_eval_invariants_and_all_tiny_placements():
    cfg = tracegen.scaled(tracegen.get_config(1), N=256, N_eval=256)
    idx, fam = tracegen.gen_trace(cfg, eval_trace=True)
    idx, fam = idx.numpy(), fam.numpy()
    L, N, k = idx.shape
    count = 0
    for pl in ref.enumerate_placements(cfg.E, cfg.P, cfg.capacity, labelled=True):
        count += 1
        if count % 9 != 1:       # every 9th of the 2520 labelled placements keeps this test quick
            continue
        primary = np.array([pl])
        out = ref.eval_placement(idx, fam, cfg.E, cfg.F, cfg.P, primary)
        # independent set-based evaluator
        span = rem = 0
        load = [0] * cfg.P
        for t in range(N):
            cards = {pl[e] for e in idx[0, t]}
            span += max(0, len(cards) - 1)
            rem += len(cards - {t % cfg.P})
            for e in idx[0, t]:
                load[pl[e]] += 1
        assert int(out["comm_span"].sum()) == span and int(out["comm_remote"].sum()) == rem
        assert out["load"][0].tolist() == load and sum(load) == N * k
        d = out["cost"][0] - np.array([max(0, len({pl[e] for e in idx[0, t]}) - 1) for t in range(N)])
        assert set(np.unique(d)) <= {0, 1}                       # comm_remote - comm_span in {0,1} per token
    assert count == 2520


def test_eval_r0_independent_of_B_theta_rho_and_P1():
    cfg, idx, fam = _small_trace(seed=23, N=200)
    primary = tracegen.random_placement(cfg.E, 4, 3, idx.shape[0], seed=1).astype(np.int64)
    a = ref.eval_placement(idx, fam, cfg.E, cfg.F, 4, primary, None, theta=0.0, rho=0.5, microbatch=7)
    b = ref.eval_placement(idx, fam, cfg.E, cfg.F, 4, primary, np.full((idx.shape[0], cfg.E, 2), -1), theta=9.0, rho=0.9, microbatch=50)
    for key in ("load", "comm_span", "comm_remote", "serve", "cost"):
        assert (a[key] == b[key]).all()
    for l in range(idx.shape[0]):
        assert (a["serve"][l] == primary[l][idx[l]]).all()
    one = ref.eval_placement(idx, fam, cfg.E, cfg.F, 1, np.zeros_like(primary), None)
    assert one["comm_span"].sum() == 0 and one["comm_remote"].sum() == 0


def test_comm_closed_form_matches_paper_baseline():
    """Pins the Comm definition (Q15): closed form under uniform routing vs the paper's printed
    Baseline Comm; then the oracle's comm_span against the same closed form (statistical)."""
    rows = []
    with open("tests/golden/paper_baseline_comm.txt") as fh:
        for line in fh:
            line = line.split("#", 1)[0].split()
            if line:
                rows.append((line[0], int(line[1]), int(line[2]), int(line[3]), int(line[4]), float(line[5])))
    for name, E, k, L, P, printed in rows:
        caps = [E // P + (1 if m < E % P else 0) for m in range(P)]
        closed = L * (sum(1 - math.comb(E - c, k) / math.comb(E, k) for c in caps) - 1)
        assert abs(closed - printed) / printed < 0.05, (name, closed, printed)
        assert printed > L                                      # the indicator reading could never exceed L
    # oracle on uniform random routing, E=64 k=6 P=16 cap 4 (one layer)
    E, k, P, cap, N = 64, 6, 16, 4, 4000
    rng = np.random.default_rng(0)
    idx = np.stack([rng.permutation(E)[:k] for _ in range(N)])[None]
    fam = np.zeros(N, dtype=np.int64)
    primary = ref.default_placement(E, cap)[None]
    out = ref.eval_placement(idx, fam, E, 1, P, primary)
    closed1 = P * (1 - math.comb(E - cap, k) / math.comb(E, k)) - 1
    assert abs(out["comm_span"].sum() / N - closed1) < 0.05      # ~4.316; sd of mean ~0.015


def test_gesr_rules():
    E, P, k = 6, 4, 3
    primary = np.array([[0, 0, 1, 2, 3, 3]])
    replicas = np.full((1, E, 2), -1)
    replicas[0, 0] = [2, 3]            # expert 0: candidates (0, 2, 3)
    idx = np.array([[[0, 2, 3], [0, 4, 5], [1, 2, 0]]])
    fam = np.zeros(3, dtype=np.int64)
    # theta = +inf: pure locality-then-load.  t0: home 0, R={1,2}: cand 0 is home, cand 2 in R -> tie on
    # locality, equal loads -> slot -> primary 0.
    S = np.zeros((1, P))
    sv = ref.gesr_select(idx, E, P, primary, replicas, S, float("inf"))
    assert sv[0, 0].tolist() == [0, 1, 2]
    # t1: home 1, R={3}: cand 3 local, others not -> 3
    assert sv[0, 1].tolist() == [3, 3, 3]
    # t2: home 2, forced R={0,1}: cand 0 in R, cand 2 = home, cand 3 not -> tie 0 vs 2 by load then slot
    assert sv[0, 2].tolist() == [0, 1, 0]
    S2 = np.array([[5.0, 0.0, 1.0, 0.0]])
    sv = ref.gesr_select(idx, E, P, primary, replicas, S2, float("inf"))
    assert sv[0, 2].tolist() == [0, 1, 2]                        # lower snapshot load wins among local
    # guard: S2 mean 1.5, thr (theta=0) 1.5 -> feas = [F,T,T,T]; t0: cand 0 infeasible -> 2 (in R)
    sv = ref.gesr_select(idx, E, P, primary, replicas, S2, 0.0)
    assert sv[0, 0].tolist() == [2, 1, 2]
    # fallback: every candidate of expert 0 infeasible -> full candidate set
    S3 = np.array([[9.0, 0.0, 9.0, 9.0]])                        # mean 6.75; feas only partition 1
    sv = ref.gesr_select(idx, E, P, primary, replicas, S3, 0.0)
    assert sv[0, 0].tolist() == [0, 1, 2]                        # same as unguarded choice
    # serve always in candidate set; chosen feasible if any feasible
    rng = np.random.default_rng(5)
    for _ in range(50):
        S = rng.random((1, P)) * 10
        feas = ref.load_guard(S[0], 0.15)
        sv = ref.gesr_select(idx, E, P, primary, replicas, S, 0.15)
        for t in range(3):
            for j in range(k):
                e = idx[0, t, j]
                cands = [primary[0, e]] + [c for c in replicas[0, e] if c >= 0]
                assert sv[0, t, j] in cands
                if len(cands) > 1 and any(feas[c] for c in cands):
                    assert feas[sv[0, t, j]]


def test_ema_special_cases():
    cfg, idx, fam = _small_trace(seed=29, N=120, L=1)
    P = 4
    primary = tracegen.random_placement(cfg.E, P, 3, 1, seed=2).astype(np.int64)
    replicas = tracegen.random_replicas(primary.astype(np.int8), P, 2, 4, seed=3).astype(np.int64)
    B = 32
    full = ref.eval_placement(idx, fam, cfg.E, cfg.F, P, primary, replicas, theta=1e9, rho=1.0, microbatch=B)
    assert np.allclose(full["load_state"], full["load"].astype(float))            # rho=1: state = cumulative load
    z = ref.eval_placement(idx, fam, cfg.E, cfg.F, P, primary, replicas, theta=0.15, rho=0.0, microbatch=B)
    last = np.zeros(P)
    for j in range(cfg.k):
        for t in range(96, 120):
            last[z["serve"][0, t, j]] += 1
    assert np.allclose(z["load_state"][0], last)                                   # rho=0: state = last Delta
    assert full["load"].sum() == 120 * cfg.k


# ---------------------------------------------------------------- fairness (O11)
def test_fairness_closed_forms():
    for P in (2, 5, 16):
        assert ref.fairness([7] * P) == (1.0, 0.0, 0.0)
        j, mv, cv = ref.fairness([0] * (P - 1) + [9])
        assert abs(j - 1.0 / P) < 1e-15 and abs(mv - (P - 1)) < 1e-12
        assert abs(cv - math.sqrt(P - 1)) < 1e-12
    assert ref.fairness([0, 0, 0]) == (1.0, 0.0, 0.0)
    L = np.random.default_rng(2).integers(1, 1000, size=16)
    j, mv, cv = ref.fairness(L)
    assert 1.0 / 16 <= j <= 1.0
    assert abs(j - L.sum() ** 2 / (16 * (L.astype(float) ** 2).sum())) < 1e-15
    assert abs(mv - (L.max() - L.mean()) / L.mean()) < 1e-15 and abs(cv - L.std() / L.mean()) < 1e-15
    assert abs(j - 1.0 / (1.0 + cv * cv)) < 1e-12                   # Jain = 1/(1+CV^2), textbook identity


# ---------------------------------------------------------------- replica table / plausibility
def test_replica_table_and_comm_reduction_plausibility():
    cfg = tracegen.scaled(tracegen.get_config(2), N=3000, N_eval=1500, L=1)
    params = tracegen.make_params(cfg)
    idx, fam = tracegen.gen_trace(cfg, params)
    from oracle import cbind
    D, C, ntok = cbind.coact(idx.numpy(), fam.numpy(), cfg.E, cfg.F)
    pr = ref.preferences(D[0].astype(np.int64), C[0].astype(np.int64), ntok.astype(np.int64))
    Abar, _, _, W = ref.graph(C[0].astype(np.int64), ntok.astype(np.int64), pr["pref"])
    primary, nsw = ref.local_search(W, cfg.P, cfg.capacity)
    assert nsw > 0 and max(Counter(primary.tolist()).values()) == cfg.capacity
    eidx, efam = tracegen.gen_trace(cfg, params, eval_trace=True)
    base = cbind.eval_placement(eidx.numpy(), efam.numpy(), cfg.E, cfg.F, cfg.P, ref.default_placement(cfg.E, cfg.capacity)[None])
    ours = cbind.eval_placement(eidx.numpy(), efam.numpy(), cfg.E, cfg.F, cfg.P, primary[None])
    assert ours["comm_span"].sum() < base["comm_span"].sum()        # Eq. 16 > 0 on planted-group traces
    aff = ref.affinity(W, primary, cfg.P)
    rep = ref.replica_table(Abar, aff, primary, n_rep=3, r=2)
    cent = Abar.sum(axis=1)
    chosen = [e for e in range(cfg.E) if rep[e, 0] >= 0]
    assert len(chosen) == 3 and set(chosen) == set(np.argsort(-cent, kind="stable")[:3].tolist())
    for e in chosen:
        assert primary[e] not in rep[e] and len(set(rep[e])) == 2
        others = [m for m in range(cfg.P) if m != primary[e]]
        assert aff[e, rep[e, 0]] == max(aff[e, m] for m in others)


# --------------------------------------------------------------------------- O13 GESR scoring (Eq. 11)
def test_gesr_scores_handworked_and_special_cases():
    # hand-worked: E=3, F=2, N_f=1.  Expert 0 co-activates with expert 1 in family 0 and with
    # expert 2 in family 1: profiles (0,1,0) and (0,0,1), mean (0,.5,.5).
    C = np.zeros((2, 3, 3), dtype=np.int64)
    C[0, 0, 1] = C[0, 1, 0] = 1
    C[1, 0, 2] = C[1, 2, 0] = 1
    s = ref.gesr_scores(C, np.array([1, 1]), lam1=2.0, lam2=3.0)
    assert s["cent"][0] == pytest.approx(1.0)                       # .5 + .5
    assert s["cons"][0] == pytest.approx(0.5 / math.sqrt(0.5))      # both cosines = .5 / (1 * sqrt(.5))
    assert s["spec"][0] == pytest.approx(math.sqrt(0.5))            # ||(0,.5,-.5)||
    assert s["score"][0] == pytest.approx(1.0 + 2.0 * math.sqrt(0.5) - 3.0 * math.sqrt(0.5))
    # expert 1: profiles (1,0,0) and (0,0,0): mean (.5,0,0); cosines 1 and 0 (zero vector, reading Q29)
    assert s["cent"][1] == pytest.approx(0.5)
    assert s["cons"][1] == pytest.approx(0.5)
    assert s["spec"][1] == pytest.approx(0.5)
    # identical families (C^f proportional to N_f): consistency 1, no specificity, any lambda
    rng = np.random.default_rng(3)
    B = rng.integers(1, 9, size=(5, 5)); B = B + B.T; np.fill_diagonal(B, 0)
    Cs = np.stack([B * 2, B * 6, B * 10])
    s = ref.gesr_scores(Cs, np.array([2, 6, 10]), lam1=0.7, lam2=0.3)
    assert np.allclose(s["cons"], 1.0, atol=1e-12) and np.allclose(s["spec"], 0.0, atol=1e-12)
    assert np.allclose(s["cent"], B.sum(axis=1), atol=1e-12)
    assert np.allclose(s["score"], s["cent"] + 0.7)
    # scaling every count by 4 (same N_f): Cent and Spec scale by 4, Cons does not move
    Cr = rng.integers(0, 7, size=(3, 6, 6)); Cr = Cr + Cr.transpose(0, 2, 1)
    for f in range(3):
        np.fill_diagonal(Cr[f], 0)
    a = ref.gesr_scores(Cr, np.array([5, 7, 9]), 0.0, 0.0)
    b = ref.gesr_scores(Cr * 4, np.array([5, 7, 9]), 0.0, 0.0)
    assert np.allclose(b["cent"], 4 * a["cent"]) and np.allclose(b["spec"], 4 * a["spec"])
    assert np.allclose(b["cons"], a["cons"])
    # an expert that is never routed: all three terms are 0
    Cz = Cr.copy(); Cz[:, 2, :] = 0; Cz[:, :, 2] = 0
    z = ref.gesr_scores(Cz, np.array([5, 7, 9]), 1.0, 1.0)
    assert z["cent"][2] == 0.0 and z["cons"][2] == 0.0 and z["spec"][2] == 0.0
    # Cauchy-Schwarz / triangle bounds that any correct implementation satisfies
    assert (a["cons"] <= 1.0 + 1e-12).all() and (a["cons"] >= 0.0).all() and (a["spec"] >= 0.0).all()


def test_gesr_replica_table_reduces_to_centrality_at_lambda_zero():
    rng = np.random.default_rng(8)
    E, F, P, cap = 12, 3, 4, 3
    Cr = rng.integers(0, 9, size=(F, E, E)); Cr = Cr + Cr.transpose(0, 2, 1)
    for f in range(F):
        np.fill_diagonal(Cr[f], 0)
    ntok = np.array([11, 13, 17])
    Abar = sum(Cr[f] / ntok[f] for f in range(F)) / F
    primary = np.arange(E) // cap
    aff = ref.affinity(Abar, primary, P)
    s = ref.gesr_scores(Cr, ntok, 0.0, 0.0)
    assert np.allclose(s["score"], Abar.sum(axis=1))
    got = ref.gesr_replica_table(s["score"], aff, primary, n_rep=4, r=2)
    assert (got == ref.replica_table(Abar, aff, primary, n_rep=4, r=2)).all()
    # structure of Eq. 12: exactly n_rep rows filled, never the primary, no duplicate partition
    filled = [e for e in range(E) if got[e, 0] >= 0]
    assert len(filled) == 4
    for e in filled:
        assert primary[e] not in got[e] and len(set(got[e])) == 2
    # a large specificity penalty removes the most family-specific expert from the generic set
    spec_top = int(np.argmax(s["spec"]))
    pen = ref.gesr_scores(Cr, ntok, 0.0, 1e6)
    rep_pen = ref.gesr_replica_table(pen["score"], aff, primary, n_rep=4, r=2)
    assert rep_pen[spec_top, 0] == -1


# ---------------------------------------------------------------------------------------------
# O14 -- spectral-then-repair grouping
# ---------------------------------------------------------------------------------------------
def _sym(E, entries):
    S = np.zeros((E, E))
    for (i, j), v in entries.items():
        S[i, j] = S[j, i] = v
    return S


def test_spectral_embedding_closed_forms():
    # scale: symmetrise then divide by the largest entry
    assert (ref.scaled_affinity(np.array([[0.0, 2.0], [4.0, 0.0]])) == np.array([[0.0, 1.0], [1.0, 0.0]])).all()
    assert (ref.scaled_affinity(np.zeros((3, 3))) == 0).all()
    # two disjoint cliques K3 + K4, no jitter: L_sym of K_n has eigenvalues 0 and n/(n-1) (n-1 times)
    W = np.zeros((7, 7))
    W[:3, :3] = 1.0
    W[3:, 3:] = 1.0
    np.fill_diagonal(W, 0.0)
    X, vals = ref.spectral_embedding(W, 7, jitter=0.0)
    assert np.allclose(vals, [0, 0, 4 / 3, 4 / 3, 4 / 3, 1.5, 1.5], atol=1e-12)
    # the null space is spanned by the (degree-weighted) clique indicators: rows equal inside a clique
    assert np.allclose(X[:3, :2], X[0, :2], atol=1e-10) and np.allclose(X[3:, :2], X[3, :2], atol=1e-10)
    assert np.linalg.norm(X[0, :2] - X[3, :2]) > 0.1
    # a path 0-1-2: L_sym eigenvalues 0, 1, 2 (bipartite)
    _, vals = ref.spectral_embedding(_sym(3, {(0, 1): 1.0, (1, 2): 1.0}), 3, jitter=0.0)
    assert np.allclose(vals, [0, 1, 2], atol=1e-12)


def test_kmeans_separated_points_and_rotation():
    rng = np.random.default_rng(3)
    truth = np.array([0, 1, 2] * 5)
    X = np.stack([truth * 10.0 + 0.1 * rng.standard_normal(15), 0.1 * rng.standard_normal(15)], axis=1)
    lab = ref.kmeans_labels(X, 3, first=0)
    assert len(set(lab)) == 3 and all((lab[i] == lab[j]) == (truth[i] == truth[j]) for i in range(15) for j in range(15))
    assert lab[0] == 0                                       # cluster ids follow the order the centres were chosen
    th = 0.7
    Q = np.array([[np.cos(th), -np.sin(th)], [np.sin(th), np.cos(th)]])
    assert ref.kmeans_labels(X @ Q, 3, first=0) == lab       # distances only: the basis does not matter
    assert ref.kmeans_labels(-X, 3, first=0) == lab
    # k = 1 and k = number of points
    assert ref.kmeans_labels(X, 1, first=4) == [0] * 15
    assert sorted(ref.kmeans_labels(X[:3], 3, first=1)) == [0, 1, 2]


def test_capacity_repair_handworked():
    # group 0 = {0,1,2,3} over capacity 3: intra sums 1.8, 1.6, 1.7, 0.7 -> expert 3 leaves and can only go to group 1
    S = _sym(5, {(0, 1): 0.9, (0, 2): 0.8, (0, 3): 0.1, (1, 2): 0.5, (1, 3): 0.2, (2, 3): 0.4, (0, 4): 0.05, (3, 4): 0.6})
    assert ref.capacity_repair(S, [0, 0, 0, 0, 1], 2, 3) == [0, 0, 0, 1, 1]
    # capacity 2: intra sums 1.7, 1.5, 1.2, 0.6 -> pool = [2, 3], strongest first.  Expert 2 prefers group 2
    # (0.7 > 0.1) and fills it; expert 3 would prefer group 2 (0.9) but only group 1 is open.
    S = _sym(6, {(0, 1): 1.0, (0, 2): 0.5, (0, 3): 0.2, (1, 2): 0.4, (1, 3): 0.1, (2, 3): 0.3,
                 (2, 4): 0.1, (2, 5): 0.7, (3, 4): 0.2, (3, 5): 0.9})
    assert ref.capacity_repair(S, [0, 0, 0, 0, 1, 2], 3, 2) == [0, 0, 2, 1, 1, 2]
    # ties: equal gains -> lower group id; equal intra sums -> lower expert id stays
    S = _sym(4, {(0, 1): 1.0, (0, 2): 1.0, (1, 2): 1.0})
    assert ref.capacity_repair(S, [0, 0, 0, 1], 3, 2) == [0, 0, 1, 1]
    # feasible input is returned unchanged
    assert ref.capacity_repair(S, [2, 0, 1, 0], 3, 2) == [2, 0, 1, 0]


def test_spectral_place_planted_and_close_to_exhaustive():
    # planted equal-size communities are recovered exactly and are the brute-force optimum of Eq. 9
    for E, P, cap, seed in ((8, 2, 4, 0), (9, 3, 3, 1), (12, 3, 4, 2)):
        rng = np.random.default_rng(seed)
        lab = np.empty(E, dtype=int)
        lab[rng.permutation(E)] = np.arange(E) // cap
        W = 0.02 * rng.random((E, E))
        W = (W + W.T) / 2 + (lab[:, None] == lab[None, :])
        np.fill_diagonal(W, 0.0)
        pr, labels0, X = ref.spectral_place(W, P, cap)
        assert X.shape == (E, P)
        assert all((pr[i] == pr[j]) == (lab[i] == lab[j]) for i in range(E) for j in range(E))
        assert pr == labels0                                 # nothing to repair
        if E <= 9:
            best, _, _ = ref.brute_force_optimum(W, P, cap)
            assert abs(ref.objective_half(W, pr) - best) < 1e-12
    # unstructured graphs: feasible, never above the optimum, and "very close to exhaustive search"
    ratios = []
    for seed in range(12):
        rng = np.random.default_rng(100 + seed)
        E, P, cap = (8, 2, 4) if seed % 2 else (9, 3, 3)
        W = rng.random((E, E)) ** 3
        W = (W + W.T) / 2
        np.fill_diagonal(W, 0.0)
        pr, _, _ = ref.spectral_place(W, P, cap)
        assert np.bincount(pr, minlength=P).max() <= cap and min(pr) >= 0
        best, _, _ = ref.brute_force_optimum(W, P, cap)
        ratios.append(ref.objective_half(W, pr) / best)
    assert max(ratios) <= 1.0 + 1e-12 and min(ratios) > 0.8 and np.mean(ratios) > 0.93
    # capacity slack (E < P*capacity): capacities are upper bounds
    W = np.random.default_rng(5).random((10, 10))
    pr, _, _ = ref.spectral_place(W, 4, 3)
    assert np.bincount(pr, minlength=4).max() <= 3


# ---------------------------------------------------------------------------------------------
# O15 -- motivation diagnostics
# ---------------------------------------------------------------------------------------------
def test_family_divergence_handworked_and_library():
    # hand-worked: E = 4, two families, one layer
    C = np.zeros((1, 2, 4, 4), dtype=np.int64)

    def put(f, i, j, v):
        C[0, f, i, j] = C[0, f, j, i] = v

    put(0, 0, 1, 5); put(0, 2, 3, 5); put(0, 0, 2, 1)           # family 0: (0,1)=5 (2,3)=5 (0,2)=1
    put(1, 0, 1, 2); put(1, 1, 3, 7)                            # family 1: (1,3)=7 (0,1)=2
    assert ref.top_pairs(C[0, 0], 2) == [(0, 1), (2, 3)]        # equal counts: smaller (i,j) first
    assert ref.top_pairs(C[0, 0], 64) == [(0, 1), (2, 3), (0, 2)]   # never a pair that did not co-activate
    assert ref.top_pairs(C[0, 1], 1) == [(1, 3)]
    D = np.array([[[4, 2, 2, 0], [1, 3, 0, 4]]], dtype=np.int64)
    ntok = np.array([4, 8], dtype=np.int64)
    frob, jac = ref.family_divergence(D, C, ntok, topk=2)
    # P0 = (1, .5, .5, 0), P1 = (.125, .375, 0, .5): squared differences .765625 + .015625 + .25 + .25
    assert abs(frob[0, 0, 1] - np.sqrt(1.28125)) < 1e-15 and frob[0, 0, 0] == 0 and frob[0, 0, 1] == frob[0, 1, 0]
    assert (frob[1] == frob[0]).all()                           # one layer: the matrix norm is the row norm
    # top-2 sets {(0,1),(2,3)} and {(1,3),(0,1)}: 1 common of 3
    assert abs(jac[0, 0, 1] - 1 / 3) < 1e-15 and jac[0, 0, 0] == 1.0 and jac[0, 1, 1] == 1.0
    # against library routines on a random case: matrix Frobenius norm, argsort-based top sets
    rng = np.random.default_rng(11)
    L, F, E, k = 3, 3, 9, 7
    D = rng.integers(0, 50, size=(L, F, E))
    ntok = rng.integers(1, 40, size=F)
    C = rng.integers(0, 6, size=(L, F, E, E))
    C = np.triu(C, 1)
    C = C + C.transpose(0, 1, 3, 2)
    frob, jac = ref.family_divergence(D, C, ntok, topk=k)
    Pm = D / ntok[None, :, None]
    for f in range(F):
        for g in range(F):
            assert abs(frob[L, f, g] - np.linalg.norm(Pm[:, f] - Pm[:, g], "fro")) < 1e-12
            for l in range(L):
                assert abs(frob[l, f, g] - np.linalg.norm(Pm[l, f] - Pm[l, g])) < 1e-12
    iu = np.triu_indices(E, 1)
    for l in range(L):
        sets = []
        for f in range(F):
            v = C[l, f][iu]
            order = np.argsort(-v, kind="stable")               # stable: row-major (i,j) order among equals
            sets.append({(int(iu[0][t]), int(iu[1][t])) for t in order[:k] if v[t] > 0})
        for f in range(F):
            for g in range(F):
                u = len(sets[f] | sets[g])
                assert abs(jac[l, f, g] - (len(sets[f] & sets[g]) / u if u else 0.0)) < 1e-15
    assert np.allclose(jac[L], jac[:L].mean(axis=0))
    # identical families: distance 0, overlap 1; a family with no tokens: empty set, overlap 0 with everything
    D2 = np.stack([D[:, 0], D[:, 0], np.zeros_like(D[:, 0])], axis=1)
    C2 = np.stack([C[:, 0], C[:, 0], np.zeros_like(C[:, 0])], axis=1)
    frob, jac = ref.family_divergence(D2, C2, np.array([5, 5, 0]), topk=k)
    assert (frob[:, 0, 1] == 0).all() and (jac[:, 0, 1] == 1).all() and (jac[:, 2, :] == 0).all()

"""The full-size C oracle (oracle/tacg_oracle.c) against the definitional Python oracle
(oracle/ref.py) and against the hand-worked trace.  CPU only."""
import numpy as np
import pytest

from oracle import ref, cbind
import tracegen


def _case(cfg_id, N, L=None, seed=None):
    cfg = tracegen.get_config(cfg_id)
    cfg = tracegen.scaled(cfg, N=N, N_eval=N, L=min(cfg.L, L or cfg.L), microbatch=max(16, N // 5))
    params = tracegen.make_params(cfg)
    idx, fam = tracegen.gen_trace(cfg, params, seed=seed)
    return cfg, idx.numpy(), fam.numpy()


@pytest.mark.parametrize("cfg_id,N,L", [(1, 512, 1), (2, 700, 2), (3, 400, 2), (5, 300, 1)])
def test_c_counts_equal_ref(cfg_id, N, L):
    cfg, idx, fam = _case(cfg_id, N, L)
    D, C, ntok = ref.coact_counts(idx, fam, cfg.E, cfg.F)
    Dc, Cc, nc = cbind.coact(idx, fam, cfg.E, cfg.F)
    assert (Dc == D).all() and (Cc == C).all() and (nc == ntok).all()
    # += semantics
    Dc2, Cc2, nc2 = cbind.coact(idx, fam, cfg.E, cfg.F, Dc.copy(), Cc.copy(), nc.copy())
    assert (Dc2 == 2 * D).all() and (Cc2 == 2 * C).all() and (nc2 == 2 * ntok).all()


def test_c_counts_skip_rules():
    idx = np.array([[[0, 1, -1], [2, -1, 3], [1, 2, 0]]], dtype=np.int16)
    fam = np.array([0, -1, 1], dtype=np.int8)
    D, C, ntok = ref.coact_counts(idx, fam, 4, 2)
    Dc, Cc, nc = cbind.coact(idx, fam, 4, 2)
    assert (Dc == D).all() and (Cc == C).all() and (nc == ntok).all()


@pytest.mark.parametrize("cfg_id,N,L", [(1, 512, 1), (2, 600, 2), (5, 500, 1)])
def test_c_affinity_equals_ref(cfg_id, N, L):
    cfg, idx, fam = _case(cfg_id, N, L)
    D, C, ntok = ref.coact_counts(idx, fam, cfg.E, cfg.F)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, cfg.L, seed=3)
    for alpha, tau in ((0.25, 1.0), (0.0, 1.0), (1.0, 0.5)):
        out = cbind.affinity_swapgain(D, C, ntok, cfg.P, primary, alpha=alpha, tau=tau, eps=1e-6)
        for l in range(cfg.L):
            pr = ref.preferences(D[l], C[l], ntok, tau=tau, eps=1e-6)
            _, _, _, W = ref.graph(C[l], ntok, pr["pref"], alpha=alpha)
            aff = ref.affinity(W, primary[l], cfg.P)
            G = ref.swap_gains(W, aff, primary[l])
            assert np.allclose(out["pref"][l], pr["pref"], rtol=1e-9, atol=1e-12)
            assert np.allclose(out["W"][l], W, rtol=1e-9, atol=1e-13)
            assert np.allclose(out["aff"][l], aff, rtol=1e-9, atol=1e-13)
            assert np.allclose(out["gain"][l], G, rtol=0, atol=1e-12)


@pytest.mark.parametrize("cfg_id,N,L,r", [(1, 600, 1, 1), (3, 500, 2, 2), (5, 700, 1, 3), (2, 300, 2, 0)])
def test_c_eval_equals_ref(cfg_id, N, L, r):
    cfg, idx, fam = _case(cfg_id, N, L)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, cfg.L, seed=5)
    replicas = tracegen.random_replicas(primary, cfg.P, r, max(2, cfg.n_rep), seed=6) if r else None
    for theta, rho, B in ((0.15, 0.995, cfg.microbatch), (0.0, 0.5, 37), (float("inf"), 1.0, 64)):
        a = ref.eval_placement(idx, fam, cfg.E, cfg.F, cfg.P, primary, replicas, theta=theta, rho=rho,
                               microbatch=B, token_offset=3)
        b = cbind.eval_placement(idx, fam, cfg.E, cfg.F, cfg.P, primary, replicas, theta=theta, rho=rho,
                                 microbatch=B, token_offset=3, want_cost=True, want_serve=True,
                                 load_state=np.zeros((cfg.L, cfg.P)))
        assert (a["load"] == b["load"]).all() and (a["serve"] == b["serve"]).all()
        assert (a["comm_span"] == b["comm_span"]).all() and (a["comm_remote"] == b["comm_remote"]).all()
        assert (a["cost"] == b["cost"]).all() and (a["ntok"] == b["ntok"]).all()
        assert (a["load_state"] == b["load_state"]).all()            # bit-exact EMA state (Q19)
        assert np.allclose(a["fairness"], b["fairness"], rtol=1e-13, atol=0)
        # gesr_select for a non-trivial snapshot
        snap = np.random.default_rng(1).random((cfg.L, cfg.P)) * 100
        sa = ref.gesr_select(idx, cfg.E, cfg.P, primary, replicas, snap, theta, token_offset=11)
        sb = cbind.gesr_select(idx, cfg.E, cfg.P, primary, replicas, snap, theta, token_offset=11)
        assert (sa == sb).all()


def test_c_eval_state_continuation():
    """Evaluating two halves with the carried load_state equals one pass (micro-batch aligned)."""
    cfg, idx, fam = _case(3, 512, 2)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, cfg.L, seed=7)
    replicas = tracegen.random_replicas(primary, cfg.P, 2, 6, seed=8)
    full = cbind.eval_placement(idx, fam, cfg.E, cfg.F, cfg.P, primary, replicas, microbatch=64,
                                load_state=np.zeros((cfg.L, cfg.P)), want_serve=True)
    h1 = cbind.eval_placement(idx[:, :256], fam[:256], cfg.E, cfg.F, cfg.P, primary, replicas, microbatch=64,
                              load_state=np.zeros((cfg.L, cfg.P)), want_serve=True)
    h2 = cbind.eval_placement(idx[:, 256:], fam[256:], cfg.E, cfg.F, cfg.P, primary, replicas, microbatch=64,
                              load_state=h1["load_state"], token_offset=256, want_serve=True)
    assert (full["load"] == h1["load"] + h2["load"]).all()
    assert (full["load_state"] == h2["load_state"]).all()
    assert (full["serve"][:, 256:] == h2["serve"]).all()


def test_c_handworked(golden_trace):
    g = golden_trace
    fam = np.array(g["family"][0], dtype=np.int8)
    idx = np.array(g["experts"], dtype=np.int16)[None]
    D, C, ntok = cbind.coact(idx, fam, 4, 2)
    assert D[0, 0].tolist() == g["D0"][0] and D[0, 1].tolist() == g["D1"][0]
    primary = np.array(g["primary"], dtype=np.int8)
    out = cbind.affinity_swapgain(D, C, ntok, 2, primary, alpha=0.25, tau=1.0, eps=1e-6)
    assert np.allclose(out["pref"][0], np.array(g["pref"]), atol=1.5e-6)
    assert np.allclose(out["W"][0], np.array(g["W"]), atol=1.5e-6)
    assert np.allclose(out["aff"][0], np.array(g["aff"]), atol=1.5e-6)
    rep = np.array(g["gesr_replicas"], dtype=np.int8)[None]
    ev = cbind.eval_placement(idx, fam, 4, 2, 2, primary, rep, theta=0.15, rho=0.995, microbatch=4,
                              load_state=np.zeros((1, 2)), want_serve=True)
    assert ev["serve"][0].tolist() == [[int(x) for x in r] for r in g["gesr_serve"]]
    assert ev["load"][0].tolist() == g["gesr_load"][0]
    assert np.allclose(ev["load_state"][0], g["gesr_state_final"][0], atol=1e-12)

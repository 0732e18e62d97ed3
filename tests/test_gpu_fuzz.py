"""Seeded random shapes through all four calls against the C oracle: small and awkward sizes
(E not a multiple of anything, F = 1, P = 1, N below one tile, more layers than SMs / fewer tokens
than CTAs, empty slots, padding tokens), every co-activation path the shape admits."""
import numpy as np
import pytest
import torch

import tracegen
from oracle import cbind

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tacg():
    import paper_2606_01007_b200 as t
    return t


@pytest.fixture(scope="module")
def ctx(tacg):
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    c = tacg.Context(0)
    yield c
    c.close()


def _case(rng):
    k = int(rng.choice([1, 2, 3, 4, 6, 8, 8, 6, 5, 16]))
    E = int(rng.integers(max(k, 2), 300))
    F = int(rng.integers(1, 9))
    L = int(rng.choice([1, 1, 2, 3, 7, 40, 160]))
    N = int(rng.choice([1, 5, 31, 33, 257, 1023, 1025, 4097, 20000]))
    if L * N > 400000:
        N = max(1, 400000 // L)
    P = int(rng.integers(1, 65))
    cap = -(-E // P) + int(rng.integers(0, 3))
    r = int(rng.integers(0, 4)) if P > 1 else 0
    B = int(rng.choice([0, 1, 7, 64, 1000, 100000]))
    return E, k, F, L, N, P, cap, r, B


@pytest.mark.parametrize("seed", list(range(24)))
def test_random_shapes(tacg, ctx, seed):
    rng = np.random.default_rng(1000 + seed)
    E, k, F, L, N, P, cap, r, B = _case(rng)
    idx = np.empty((L, N, k), dtype=np.int16)
    for l in range(L):
        keys = rng.random((N, E))
        idx[l] = np.argsort(keys, axis=1)[:, :k]                     # k distinct experts per token
    idx[rng.random(idx.shape) < 0.03] = -1                           # empty slots
    fam = rng.integers(0, F, size=N).astype(np.int8)
    fam[rng.random(N) < 0.02] = -1                                   # padding tokens
    D, C, ntok = cbind.coact(idx, fam, E, F)
    di, df = torch.from_numpy(idx).cuda(), torch.from_numpy(fam).cuda()
    paths = [tacg.TACG_PATH_HIST]
    if k in (2, 4, 6, 8) and E <= 256:
        paths.append(tacg.TACG_PATH_MMA)
    for flag in paths:
        out = tacg.tacg_coact_accumulate(ctx, di, df, E, F, flags=tacg.TACG_ZERO_FIRST | flag)
        torch.cuda.synchronize()
        assert (out["D"].cpu().numpy().view(np.uint32) == D).all(), (flag, "D")
        assert (out["C"].cpu().numpy().view(np.uint32) == C).all(), (flag, "C")
        assert (out["ntok"].cpu().numpy().view(np.uint64) == ntok).all(), (flag, "ntok")
    primary = tracegen.random_placement(E, P, cap, L, seed=seed)
    replicas = tracegen.random_replicas(primary, P, r, max(1, E // 6), seed=seed + 1) if r else None
    state0 = rng.random((L, P)) * 20.0
    theta = float(rng.choice([0.0, 0.15, 1.0]))
    want = cbind.eval_placement(idx, fam, E, F, P, primary, replicas, theta=theta, rho=0.9, microbatch=B,
                                token_offset=int(seed), want_cost=True, want_serve=True, load_state=state0.copy())
    st = torch.from_numpy(state0.copy()).cuda()
    got = tacg.tacg_eval_placement(ctx, di, df, E, F, P, torch.from_numpy(primary).cuda(),
                                   None if replicas is None else torch.from_numpy(replicas).cuda(), theta=theta,
                                   rho=0.9, microbatch=B, token_offset=int(seed), load_state=st, want_cost=True,
                                   want_serve=True)
    torch.cuda.synchronize()
    assert (got["load"].cpu().numpy().view(np.uint64) == want["load"]).all()
    assert (got["comm_span"].cpu().numpy().view(np.uint64) == want["comm_span"]).all()
    assert (got["comm_remote"].cpu().numpy().view(np.uint64) == want["comm_remote"]).all()
    assert (got["ntok"].cpu().numpy().view(np.uint64) == want["ntok"]).all()
    assert (got["cost"].cpu().numpy() == want["cost"]).all()
    assert (got["serve"].cpu().numpy() == want["serve"]).all()
    assert (st.cpu().numpy().view(np.uint64) == want["load_state"].view(np.uint64)).all()
    assert np.allclose(got["fairness"].cpu().numpy().astype(np.float64), want["fairness"], rtol=1e-5, atol=1e-7)
    if replicas is not None:
        snap = rng.random((L, P)) * 30.0
        sv = tacg.gesr_select(ctx, di, E, P, torch.from_numpy(primary).cuda(), torch.from_numpy(replicas).cuda(),
                              torch.from_numpy(snap).cuda(), theta, token_offset=2)
        assert (sv.cpu().numpy() == cbind.gesr_select(idx, E, P, primary, replicas, snap, theta, 2)).all()


@pytest.mark.parametrize("seed", list(range(16)))
def test_random_shapes_offline_stage(tacg, ctx, seed):
    """The E x E kernels on awkward shapes: the cluster-fused affinity kernel (every family count 1..8, E not a
    multiple of the 8-row blocks or of the cluster's 64 rows, more layers than clusters fit), the GESR offline step,
    the capacity repair and the divergence diagnostics, against the oracle."""
    from oracle import ref
    rng = np.random.default_rng(5000 + seed)
    k = int(rng.choice([2, 4, 6, 8, 3]))
    E = int(rng.integers(max(k, 3), 200))
    F = int(rng.integers(1, 9))
    L = int(rng.choice([1, 2, 3, 21]))
    N = int(rng.choice([300, 2000, 6000]))
    P = int(rng.integers(2, min(E, 64) + 1))
    cap = -(-E // P) + int(rng.integers(0, 3))
    idx = np.empty((L, N, k), dtype=np.int16)
    hot = rng.dirichlet(np.full(E, 0.3), size=(L, F))                # family-dependent popularity, so sigma > 0
    fam = rng.integers(0, F, size=N).astype(np.int8)
    for l in range(L):
        keys = rng.random((N, E)) ** (1.0 / np.maximum(hot[l][fam], 1e-9))
        idx[l] = np.argsort(-keys, axis=1)[:, :k]
    D, C, ntok = cbind.coact(idx, fam, E, F)
    primary = tracegen.random_placement(E, P, cap, L, seed=seed)
    alpha, tau = float(rng.choice([0.0, 0.25, 0.6])), float(rng.choice([0.5, 1.0, 2.0]))
    want = cbind.affinity_swapgain(D, C, ntok, P, primary, alpha=float(np.float32(alpha)), tau=float(np.float32(tau)),
                                   eps=float(np.float32(1e-6)))
    dD = torch.from_numpy(D.view(np.int32)).cuda()
    dC = torch.from_numpy(C.view(np.int32)).cuda()
    dn = torch.from_numpy(ntok.view(np.int64)).cuda()
    dp = torch.from_numpy(primary).cuda()
    got = tacg.tacg_affinity_swapgain(ctx, dD, dC, dn, P, cap, dp, alpha=alpha, tau=tau, eps=1e-6)
    torch.cuda.synchronize()
    for key in ("pref", "W", "aff"):
        g = got[key].cpu().numpy().astype(np.float64)
        assert (np.abs(g - want[key]) <= 1e-5 * np.maximum(np.abs(want[key]), 1e-6)).all(), key
    G = got["gain"].cpu().numpy().astype(np.float64)
    for l in range(L):
        pr = primary[l].astype(np.int64)
        aff, W = want["aff"][l], want["W"][l]
        ia, ib = aff[np.arange(E), pr], aff[:, pr]
        mag = np.abs(ib) + np.abs(ib.T) + np.abs(ia)[:, None] + np.abs(ia)[None, :] + 2 * np.abs(W)
        assert (np.abs(G[l] - want["gain"][l]) <= 1e-5 * np.maximum(mag, 1e-6)).all(), ("gain", l)
    # W alone (no placement): the kernel leaves before the affinity phases
    only_w = tacg.tacg_affinity_swapgain(ctx, dD, dC, dn, P, cap, None, alpha=alpha, tau=tau, eps=1e-6, want=("W",))["W"]
    assert torch.equal(only_w, got["W"])
    # GESR offline terms
    _, terms = tacg.gesr_build_replicas(ctx, dD, dC, dn, P, cap, dp, max(1, E // 8), min(2, P - 1), lambda1=0.5,
                                        lambda2=0.25, alpha=alpha, tau=tau)
    sc = ref.gesr_scores(C[0].astype(np.int64), ntok, 0.5, 0.25)
    t0 = terms[0].cpu().numpy().astype(np.float64)
    for col, key in enumerate(("score", "cent", "cons", "spec")):
        assert np.allclose(t0[:, col], sc[key], rtol=1e-5, atol=1e-9), key
    # capacity repair from skewed labels: exact
    Wh = np.ascontiguousarray(want["W"], dtype=np.float32)
    labels = np.minimum(rng.geometric(0.4, size=(L, E)) - 1, P - 1).astype(np.int8)
    rep = tacg.tacg_spectral_place(ctx, torch.from_numpy(Wh).cuda(), P, cap, labels_in=torch.from_numpy(labels).cuda())
    for l in range(min(L, 3)):
        assert rep["primary"][l].cpu().numpy().tolist() == ref.capacity_repair(ref.scaled_affinity(Wh[l]), labels[l], P, cap)
    # divergence diagnostics on the first layers
    Ls = min(L, 2)
    fr, jc = tacg.tacg_family_divergence(ctx, dD[:Ls].contiguous(), dC[:Ls].contiguous(), dn, topk=64)
    wf, wj = ref.family_divergence(D[:Ls].astype(np.int64), C[:Ls].astype(np.int64), ntok.astype(np.int64), topk=64)
    assert (jc[:-1].cpu().numpy() == wj[:-1].astype(np.float32)).all()
    assert np.allclose(fr.cpu().numpy().astype(np.float64), wf, rtol=1e-6, atol=1e-12)

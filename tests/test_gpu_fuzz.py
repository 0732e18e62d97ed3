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

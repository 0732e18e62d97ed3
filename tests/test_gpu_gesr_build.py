"""gesr_build_replicas against the oracle: Eq. 11 terms within 1e-5 relative;
the replica table exactly, except where the oracle's own ranking is a near-tie (two fp64 scores or
affinities closer than 1e-9 relative), in which case either order is accepted and only the unique
part is compared."""
import numpy as np
import pytest
import torch

import tracegen
from oracle import cbind, ref

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


def _near_tie(values, n):
    """True when the n-th and (n+1)-th largest values are closer than 1e-9 relative."""
    v = np.sort(np.asarray(values, dtype=np.float64))[::-1]
    if n <= 0 or n >= len(v):
        return False
    return abs(v[n - 1] - v[n]) <= 1e-9 * max(abs(v[n - 1]), 1e-300)


@pytest.mark.parametrize("cfg_id,N,L,n_rep,r,lam1,lam2", [
    (1, 4096, 1, 2, 1, 0.0, 0.0), (2, 30000, 3, 6, 2, 0.0, 0.0), (2, 30000, 2, 6, 2, 0.5, 0.25),
    (3, 20000, 2, 4, 2, 1.0, 0.1), (5, 40000, 1, 5, 3, 2.0, 1.0), (4, 12000, 2, 8, 2, 0.25, 0.05),
])
def test_gesr_build_matches_oracle(tacg, ctx, cfg_id, N, L, n_rep, r, lam1, lam2):
    cfg = tracegen.scaled(tracegen.get_config(cfg_id), N=N, N_eval=N, L=min(L, tracegen.get_config(cfg_id).L))
    params = tracegen.make_params(cfg)
    idx, fam = tracegen.gen_trace(cfg, params)
    D, C, ntok = cbind.coact(idx.numpy(), fam.numpy(), cfg.E, cfg.F)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, cfg.L, seed=9)
    co = tacg.tacg_coact_accumulate(ctx, idx.cuda(), fam.cuda(), cfg.E, cfg.F, flags=tacg.TACG_ZERO_FIRST)
    rep, terms = tacg.gesr_build_replicas(ctx, co["D"], co["C"], co["ntok"], cfg.P, cfg.capacity,
                                          torch.from_numpy(primary).cuda(), n_rep, r, lambda1=lam1, lambda2=lam2)
    torch.cuda.synchronize()
    rep, terms = rep.cpu().numpy(), terms.cpu().numpy().astype(np.float64)
    want_aff = cbind.affinity_swapgain(D, C, ntok, cfg.P, primary, alpha=0.25, tau=1.0, eps=float(np.float32(1e-6)))["aff"]
    for l in range(cfg.L):
        s = ref.gesr_scores(C[l].astype(np.int64), ntok, float(np.float32(lam1)), float(np.float32(lam2)))
        for col, key in enumerate(("score", "cent", "cons", "spec")):
            w = s[key]
            assert (np.abs(terms[l, :, col] - w) <= 1e-5 * np.maximum(np.abs(w), 1e-6) + 1e-12).all(), (l, key)
        want = ref.gesr_replica_table(s["score"], want_aff[l], primary[l], n_rep, r)
        got_set = {e for e in range(cfg.E) if rep[l, e, 0] >= 0}
        want_set = {e for e in range(cfg.E) if want[e, 0] >= 0}
        if not _near_tie(s["score"], n_rep):
            assert got_set == want_set, l
        assert len(got_set) == min(n_rep, cfg.E)
        for e in got_set & want_set:
            others = [want_aff[l, e, m] for m in range(cfg.P) if m != primary[l, e]]
            if any(_near_tie(others, q) for q in range(1, r + 1)):
                assert primary[l, e] not in rep[l, e] and len(set(rep[l, e])) == r
            else:
                assert (rep[l, e] == want[e]).all(), (l, e)
        for e in set(range(cfg.E)) - got_set:
            assert (rep[l, e] == -1).all()


def test_gesr_build_feeds_eval_and_errors(tacg, ctx):
    cfg = tracegen.scaled(tracegen.get_config(3), N=8000, N_eval=8000, L=2, microbatch=1024)
    params = tracegen.make_params(cfg)
    idx, fam = tracegen.gen_trace(cfg, params)
    co = tacg.tacg_coact_accumulate(ctx, idx.cuda(), fam.cuda(), cfg.E, cfg.F, flags=tacg.TACG_ZERO_FIRST)
    primary = torch.from_numpy(tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, cfg.L, seed=2)).cuda()
    rep, _ = tacg.gesr_build_replicas(ctx, co["D"], co["C"], co["ntok"], cfg.P, cfg.capacity, primary, 4, 2)
    # the table is a valid input of the evaluator (its own device-side validation accepts it)
    tacg.tacg_eval_placement(ctx, idx.cuda(), fam.cuda(), cfg.E, cfg.F, cfg.P, primary, rep, microbatch=cfg.microbatch,
                             flags=tacg.TACG_VALIDATE)
    L, F, E = co["D"].shape
    out = torch.empty((L, E, 2), dtype=torch.int8, device="cuda")
    args = (co["D"], co["C"], co["ntok"], L, E, F, cfg.P, cfg.capacity, primary, 0.25, 1.0, 1e-6, 0.0, 0.0)
    assert ctx.gesr_build_replicas(*args, 4, 0, out, None) == -2          # r < 1
    assert ctx.gesr_build_replicas(*args, -1, 2, out, None) == -2         # n_rep < 0
    assert ctx.gesr_build_replicas(*args, 4, 2, None, None) == -1         # NULL output

"""tacg_family_divergence against oracle O15.  The top-k pair sets come from
an exact integer select, so the Jaccard overlap is the oracle's rational number rounded to fp32; the
distance is an fp64 sum stored as fp32 (1e-6 relative)."""
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


def _compare(tacg, ctx, D, C, ntok, topk):
    frob, jac = tacg.tacg_family_divergence(ctx, torch.from_numpy(D.astype(np.uint32).view(np.int32)).cuda(),
                                            torch.from_numpy(C.astype(np.uint32).view(np.int32)).cuda(),
                                            torch.from_numpy(ntok.astype(np.uint64).view(np.int64)).cuda(), topk=topk)
    torch.cuda.synchronize()
    want_f, want_j = ref.family_divergence(D.astype(np.int64), C.astype(np.int64), ntok.astype(np.int64), topk=topk)
    assert (jac.cpu().numpy() == want_j.astype(np.float32)).all() or \
        np.abs(jac.cpu().numpy().astype(np.float64) - want_j).max() <= 1e-7     # row L: mean of rationals
    assert (jac[:-1].cpu().numpy() == want_j[:-1].astype(np.float32)).all()
    assert np.allclose(frob.cpu().numpy().astype(np.float64), want_f, rtol=1e-6, atol=1e-12)


@pytest.mark.parametrize("cfg_id,N,L,topk", [(1, 4096, 1, 64), (2, 30000, 3, 64), (3, 20000, 2, 64), (4, 12000, 2, 64),
                                             (5, 40000, 1, 64), (2, 3000, 2, 256), (3, 500, 2, 64), (2, 30000, 2, 1)])
def test_divergence_on_traces(tacg, ctx, cfg_id, N, L, topk):
    cfg = tracegen.scaled(tracegen.get_config(cfg_id), N=N, N_eval=N, L=min(L, tracegen.get_config(cfg_id).L))
    idx, fam = tracegen.gen_trace(cfg, tracegen.make_params(cfg))
    D, C, ntok = cbind.coact(idx.numpy(), fam.numpy(), cfg.E, cfg.F)
    _compare(tacg, ctx, D, C, ntok, topk)


@pytest.mark.parametrize("seed", range(6))
def test_divergence_heavy_ties_and_sparse_counts(tacg, ctx, seed):
    """Small count ranges make the k-th largest count a many-way tie (the ordered part of the select); sparse
    matrices have fewer than k positive pairs (the take-everything branch); one family is empty."""
    rng = np.random.default_rng(seed)
    L, F, E = 2, 4, int(rng.integers(5, 70))
    hi = int(rng.choice([2, 3, 300, 70000]))
    C = rng.integers(0, hi, size=(L, F, E, E), dtype=np.int64)
    C[rng.random(C.shape) < rng.choice([0.0, 0.9, 0.995])] = 0
    C = np.triu(C, 1)
    C = C + C.transpose(0, 1, 3, 2)
    C[:, 3] = 0
    D = rng.integers(0, 1000, size=(L, F, E), dtype=np.int64)
    D[:, 3] = 0
    ntok = np.array([int(rng.integers(1, 500)), 7, 1, 0], dtype=np.int64)
    _compare(tacg, ctx, D, C, ntok, int(rng.choice([1, 5, 64, 200])))


def test_divergence_refusals(tacg, ctx):
    D = torch.zeros((1, 2, 4), dtype=torch.int32, device="cuda")
    C = torch.zeros((1, 2, 4, 4), dtype=torch.int32, device="cuda")
    n = torch.zeros((2,), dtype=torch.int64, device="cuda")
    for topk in (0, 257):
        with pytest.raises(tacg.TacgError):
            tacg.tacg_family_divergence(ctx, D, C, n, topk=topk)
    frob, jac = tacg.tacg_family_divergence(ctx, D, C, n)
    assert (frob == 0).all() and (jac == 0).all()

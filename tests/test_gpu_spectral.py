"""tacg_spectral_place against the oracle.

Stage 2 (the repair) sums in the oracle's order in fp64, so with Stage 1 replaced by given labels
it is compared bit for bit.  Stage 1 goes through two different eigensolvers (LAPACK in the oracle,
one-sided Jacobi on the device): what is unique is compared -- the projector onto the embedding's
column space, and the labels, which depend on distances only (Q35).  Every W handed to
both sides is made on the host (the oracle's graph, or a seeded random graph).
"""
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


def _oracle_graph(cfg_id, N, L):
    cfg = tracegen.scaled(tracegen.get_config(cfg_id), N=N, N_eval=N, L=min(L, tracegen.get_config(cfg_id).L))
    params = tracegen.make_params(cfg)
    idx, fam = tracegen.gen_trace(cfg, params)
    D, C, ntok = cbind.coact(idx.numpy(), fam.numpy(), cfg.E, cfg.F)
    any_primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, cfg.L, seed=1)     # W does not depend on it
    W = cbind.affinity_swapgain(D, C, ntok, cfg.P, any_primary, alpha=0.25, tau=1.0, eps=float(np.float32(1e-6)))["W"]
    return cfg, np.ascontiguousarray(W, dtype=np.float32)


def _random_graph(L, E, seed, power=3):
    rng = np.random.default_rng(seed)
    W = rng.random((L, E, E)) ** power
    W = (W + W.transpose(0, 2, 1)) / 2
    for l in range(L):
        np.fill_diagonal(W[l], 0.0)
    return W.astype(np.float32)


@pytest.mark.parametrize("L,E,P,cap,seed", [(3, 60, 16, 8, 0), (2, 64, 8, 8, 1), (2, 160, 16, 10, 2), (1, 256, 32, 8, 3),
                                            (4, 7, 3, 3, 4), (2, 33, 5, 7, 5), (1, 512, 64, 8, 6), (2, 12, 12, 1, 7)])
def test_repair_alone_is_exact(tacg, ctx, L, E, P, cap, seed):
    W = _random_graph(L, E, seed)
    rng = np.random.default_rng(seed + 100)
    # skewed start: most experts in a few groups, so groups overflow and the pool is long
    labels = np.minimum(rng.geometric(0.35, size=(L, E)) - 1, P - 1).astype(np.int8)
    got = tacg.tacg_spectral_place(ctx, torch.from_numpy(W).cuda(), P, cap, labels_in=torch.from_numpy(labels).cuda())
    torch.cuda.synchronize()
    pr = got["primary"].cpu().numpy()
    assert (got["labels0"].cpu().numpy() == labels).all()
    for l in range(L):
        want = ref.capacity_repair(ref.scaled_affinity(W[l]), labels[l], P, cap)
        assert pr[l].tolist() == want, l
        assert np.bincount(pr[l], minlength=P).max() <= cap


def _check_full(tacg, ctx, W, P, cap):
    L, E, _ = W.shape
    got = tacg.tacg_spectral_place(ctx, torch.from_numpy(W).cuda(), P, cap, want_embed=True)
    torch.cuda.synchronize()
    pr, l0, X = got["primary"].cpu().numpy(), got["labels0"].cpu().numpy(), got["embed"].cpu().numpy()
    for l in range(L):
        want_pr, want_l0, want_X = ref.spectral_place(W[l], P, cap)
        # the embedding: orthonormal columns spanning the oracle's eigenspace
        assert np.abs(X[l].T @ X[l] - np.eye(P)).max() < 1e-9
        _, vals = ref.spectral_embedding(W[l], min(E, P + 1))
        if E == P or vals[P] - vals[P - 1] > 1e-6:         # the space is unique only with a gap above it
            assert np.abs(X[l] @ X[l].T - want_X @ want_X.T).max() < 1e-7, l
        assert l0[l].tolist() == want_l0, l
        assert pr[l].tolist() == want_pr, l
        assert np.bincount(pr[l], minlength=P).max() <= cap and pr[l].min() >= 0
    return pr


@pytest.mark.parametrize("cfg_id,N,L", [(1, 4096, 1), (2, 30000, 3), (3, 20000, 2), (5, 40000, 1), (4, 20000, 2), (4, 200000, 1)])
def test_spectral_place_on_the_methods_graph(tacg, ctx, cfg_id, N, L):
    cfg, W = _oracle_graph(cfg_id, N, L)
    pr = _check_full(tacg, ctx, W, cfg.P, cfg.capacity)
    # the point of the step: a better Eq. 9 objective than a random feasible placement
    rnd = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, cfg.L, seed=3)
    for l in range(cfg.L):
        assert ref.objective_half(W[l].astype(np.float64), pr[l]) > ref.objective_half(W[l].astype(np.float64), rnd[l])


@pytest.mark.parametrize("L,E,P,cap,seed", [(2, 8, 2, 4, 0), (3, 9, 3, 3, 1), (2, 24, 4, 6, 2), (1, 31, 4, 9, 3), (1, 96, 12, 8, 4)])
def test_spectral_place_random_and_planted(tacg, ctx, L, E, P, cap, seed):
    _check_full(tacg, ctx, _random_graph(L, E, seed), P, cap)
    rng = np.random.default_rng(seed)
    lab = np.empty(E, dtype=int)
    lab[rng.permutation(E)] = np.arange(E) % P
    W = (0.02 * _random_graph(1, E, seed + 50, power=1)[0] + (lab[:, None] == lab[None, :])).astype(np.float32)
    np.fill_diagonal(W, 0.0)
    pr = _check_full(tacg, ctx, W[None], P, cap)[0]
    if E % P == 0 and E // P <= cap:
        assert all((pr[i] == pr[j]) == (lab[i] == lab[j]) for i in range(E) for j in range(E))


def test_spectral_place_degenerate_and_refusals(tacg, ctx):
    # an all-zero graph: only the jitter is left; any feasible answer must still come back, and match the oracle
    W = np.zeros((1, 6, 6), dtype=np.float32)
    got = tacg.tacg_spectral_place(ctx, torch.from_numpy(W).cuda(), 3, 2, labels_in=torch.zeros((1, 6), dtype=torch.int8).cuda())
    assert got["primary"].cpu().numpy()[0].tolist() == ref.capacity_repair(ref.scaled_affinity(W[0]), [0] * 6, 3, 2)
    # P = 1: one group
    W = _random_graph(1, 5, 9)
    got = tacg.tacg_spectral_place(ctx, torch.from_numpy(W).cuda(), 1, 5)
    assert (got["primary"].cpu().numpy() == 0).all()
    # an expert that never co-activates (an all-zero row and column of W): isolated, still placed like the oracle places it
    W = _random_graph(1, 8, 3)
    W[0, 5, :] = 0.0
    W[0, :, 5] = 0.0
    _check_full(tacg, ctx, W, 2, 4)
    Wd = torch.from_numpy(_random_graph(1, 8, 1)).cuda()
    for P, cap, jit, iters in ((9, 1, 1e-6, 10), (2, 3, 1e-6, 10), (2, 4, -1.0, 10), (2, 4, 0.0, 10), (2, 4, 1e-6, 0), (65, 1, 1e-6, 10)):
        with pytest.raises(tacg.TacgError):
            tacg.tacg_spectral_place(ctx, Wd, P, cap, jitter=jit, kmeans_iters=iters)

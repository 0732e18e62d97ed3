"""The paper's skew sweep (section 4.3, PAPER.md:383 the 13-workload suite): one placement, thirteen online family
streams.  Only the family labels change, which is exactly what moves work between the family
bins of the counting kernels and between the per-family accumulators of the evaluator, so every
stream is a parity case for both: counts and evaluation bit-exact against the C oracle.
"""
import numpy as np
import pytest
import torch

import tracegen
from oracle import cbind

pytestmark = pytest.mark.gpu

WORKLOADS = tracegen.skew_workloads(4)


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


@pytest.fixture(scope="module")
def setup():
    cfg = tracegen.scaled(tracegen.get_config(3), L=2, N=30011, N_eval=30011)
    params = tracegen.make_params(cfg)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, cfg.L, seed=cfg.seed)
    replicas = tracegen.random_replicas(primary, cfg.P, 2, 12, seed=cfg.seed + 1)
    return cfg, params, primary, replicas


def _u32(t):
    return t.cpu().numpy().view(np.uint32)


def _u64(t):
    return t.cpu().numpy().view(np.uint64)


@pytest.mark.parametrize("workload", WORKLOADS)
def test_skew_stream_parity(tacg, ctx, setup, workload):
    cfg, params, primary, replicas = setup
    fam = tracegen.gen_family_workload(cfg.N_eval, workload, cfg.F, seed=cfg.seed + 3)
    idx = tracegen.gen_indices(cfg, params, fam, cfg.seed + 3, eval_trace=True)
    idx_d, fam_d = idx.cuda(), fam.cuda()
    wD, wC, wn = cbind.coact(idx.numpy(), fam.numpy(), cfg.E, cfg.F)
    for flag in (tacg.TACG_PATH_HIST, tacg.TACG_PATH_MMA):
        out = tacg.tacg_coact_accumulate(ctx, idx_d, fam_d, cfg.E, cfg.F, flags=tacg.TACG_ZERO_FIRST | flag)
        torch.cuda.synchronize()
        assert (_u64(out["ntok"]) == wn).all()
        assert (_u32(out["D"]) == wD).all()
        assert (_u32(out["C"]) == wC).all()
    st = torch.zeros((cfg.L, cfg.P), dtype=torch.float64, device="cuda")
    got = tacg.tacg_eval_placement(ctx, idx_d, fam_d, cfg.E, cfg.F, cfg.P, torch.from_numpy(primary).cuda(),
                                   torch.from_numpy(replicas).cuda(), theta=0.15, rho=0.995, microbatch=4096,
                                   load_state=st, want_cost=True)
    torch.cuda.synchronize()
    want = cbind.eval_placement(idx.numpy(), fam.numpy(), cfg.E, cfg.F, cfg.P, primary, replicas, theta=0.15,
                                rho=0.995, microbatch=4096, load_state=np.zeros((cfg.L, cfg.P)), want_cost=True)
    for key in ("load", "comm_span", "comm_remote", "ntok"):
        assert (_u64(got[key]) == want[key]).all(), key
    assert (got["cost"].cpu().numpy() == want["cost"]).all()
    assert (st.cpu().numpy().view(np.uint64) == want["load_state"].view(np.uint64)).all()
    assert np.allclose(got["fairness"].cpu().numpy().astype(np.float64), want["fairness"], rtol=1e-5, atol=1e-7)

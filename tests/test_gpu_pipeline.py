"""End-to-end slice on the GPU: accumulate -> W / swap gains -> host local
search -> replica table -> evaluation.  The placement driver is a consumer of the hot path; what is
checked is that it feeds the library valid inputs and that the GPU swap gains do what Eq. 9/10 say:
every applied swap raises the within-partition affinity objective computed by the oracle."""
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


def _objective(W, primary):
    """J_half = sum_{i<j, same partition} W[i,j] per layer (Eq. 9 over unordered pairs, Q11)."""
    same = primary[:, :, None] == primary[:, None, :]
    return (np.triu(W, 1) * np.triu(same, 1)).sum(axis=(1, 2))


@pytest.mark.parametrize("cfg_id,N,L", [(2, 30000, 3), (3, 20000, 2)])
def test_pipeline_local_search_and_eval(tacg, ctx, cfg_id, N, L):
    from paper_2606_01007_b200 import placement
    cfg = tracegen.scaled(tracegen.get_config(cfg_id), N=N, N_eval=N, L=L, microbatch=4096)
    params = tracegen.make_params(cfg)
    bi, bf = tracegen.gen_trace(cfg, params)
    ei, ef = tracegen.gen_trace(cfg, params, eval_trace=True)
    co = tacg.tacg_coact_accumulate(ctx, bi.cuda(), bf.cuda(), cfg.E, cfg.F, flags=tacg.TACG_ZERO_FIRST)
    base = placement.default_placement(cfg.L, cfg.E, cfg.capacity)
    primary, swaps = placement.local_search(ctx, co["D"], co["C"], co["ntok"], cfg.P, cfg.capacity)
    # capacity preserved, and the oracle's objective did not go down on any layer
    for l in range(cfg.L):
        assert np.bincount(primary[l], minlength=cfg.P).max() <= cfg.capacity
    D, C, ntok = cbind.coact(bi.numpy(), bf.numpy(), cfg.E, cfg.F)
    want = cbind.affinity_swapgain(D, C, ntok, cfg.P, base, alpha=0.25, tau=1.0, eps=float(np.float32(1e-6)))
    j0, j1 = _objective(want["W"], base), _objective(want["W"], primary)
    assert (j1 >= j0 - 1e-9).all()
    assert (j1[swaps > 0] > j0[swaps > 0]).all()
    # the replica table passes the library's own validation and the evaluation matches the oracle
    r = max(cfg.r, 1)
    replicas = tacg.gesr_build_replicas(ctx, co["D"], co["C"], co["ntok"], cfg.P, cfg.capacity,
                                        torch.from_numpy(primary).cuda(), 4, r)[0].cpu().numpy()
    got = tacg.tacg_eval_placement(ctx, ei.cuda(), ef.cuda(), cfg.E, cfg.F, cfg.P, torch.from_numpy(primary).cuda(),
                                   torch.from_numpy(replicas).cuda(), theta=0.15, rho=0.995,
                                   microbatch=cfg.microbatch, flags=tacg.TACG_VALIDATE)
    torch.cuda.synchronize()
    ref = cbind.eval_placement(ei.numpy(), ef.numpy(), cfg.E, cfg.F, cfg.P, primary, replicas, theta=0.15, rho=0.995,
                               microbatch=cfg.microbatch, load_state=np.zeros((cfg.L, cfg.P)))
    assert (got["load"].cpu().numpy().view(np.uint64) == ref["load"]).all()
    assert (got["comm_span"].cpu().numpy().view(np.uint64) == ref["comm_span"]).all()
    assert (got["comm_remote"].cpu().numpy().view(np.uint64) == ref["comm_remote"]).all()


@pytest.mark.parametrize("cfg_id,N,L", [(2, 40000, 3), (3, 30000, 2), (5, 60000, 1)])
def test_offline_stage_on_device_then_eval(tacg, ctx, cfg_id, N, L):
    """counts -> graph -> spectral-then-repair -> replicas -> evaluation, nothing computed on the host.
    The evaluation of the resulting placement is bit-exact against the oracle, and the placement does
    what the method is for: fewer partitions touched per token on a held-out trace than the paper's
    'Baseline' contiguous placement, with and without replicas."""
    from paper_2606_01007_b200 import placement
    cfg = tracegen.scaled(tracegen.get_config(cfg_id), N=N, N_eval=N, L=min(L, tracegen.get_config(cfg_id).L), microbatch=4096)
    params = tracegen.make_params(cfg)
    bi, bf = tracegen.gen_trace(cfg, params)
    ei, ef = tracegen.gen_trace(cfg, params, eval_trace=True)
    co = tacg.tacg_coact_accumulate(ctx, bi.cuda(), bf.cuda(), cfg.E, cfg.F, flags=tacg.TACG_ZERO_FIRST)
    primary, replicas = placement.tacg_gesr_placement(ctx, co["D"], co["C"], co["ntok"], cfg.P, cfg.capacity, 6, 2)
    base = torch.from_numpy(placement.default_placement(cfg.L, cfg.E, cfg.capacity)).cuda()
    spans = {}
    for name, pr, rep in (("baseline", base, None), ("tacg", primary, None), ("tacg+gesr", primary, replicas)):
        got = tacg.tacg_eval_placement(ctx, ei.cuda(), ef.cuda(), cfg.E, cfg.F, cfg.P, pr, rep, theta=0.15, rho=0.995,
                                       microbatch=cfg.microbatch, flags=tacg.TACG_VALIDATE)
        torch.cuda.synchronize()
        want = cbind.eval_placement(ei.numpy(), ef.numpy(), cfg.E, cfg.F, cfg.P, pr.cpu().numpy(),
                                    None if rep is None else rep.cpu().numpy(), theta=0.15, rho=0.995,
                                    microbatch=cfg.microbatch, load_state=np.zeros((cfg.L, cfg.P)))
        for key in ("load", "comm_span", "comm_remote", "ntok"):
            assert (got[key].cpu().numpy().view(np.uint64) == want[key]).all(), (name, key)
        spans[name] = int(want["comm_span"].sum())
    assert spans["tacg"] < spans["baseline"]
    # replicas serve under the load guard (Eq. 13), which may trade a little locality for balance
    assert spans["tacg+gesr"] < spans["baseline"]

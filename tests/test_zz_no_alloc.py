"""tacg_eval_primary_noalloc (include/tacg.h): the primary-only evaluation through the entry point that allocates
nothing -- its scratch is a fixed device array inside the library -- against tacg_eval_placement with replicas = NULL,
the existing path (itself checked against the oracle in test_gpu_parity.py / test_gpu_fullsize.py).

Integers and EMA bits are compared bit for bit, fairness within the 1e-5 of the other GPU tests; two calls in a row
(different traces and shapes, so the second call finds the first call's rows in the array), then the first again.
Also: the size limit is refused with TACG_ERR_SHAPE, and the calls leave the CUDA allocator alone.

The file sorts after every other test file: the suite runs with pytest -x, a failure here must not hide the others.
"""
import numpy as np
import pytest
import torch

import tracegen

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


def _case(cfg_id, N, L, seed, want_outputs):
    cfg = tracegen.scaled(tracegen.get_config(cfg_id), N=N, N_eval=N, L=L)
    idx, fam = tracegen.gen_trace(cfg, tracegen.make_params(cfg), eval_trace=True)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, L, seed=seed)
    return cfg, idx.cuda(), fam.cuda(), torch.from_numpy(primary).cuda(), want_outputs


def _outputs(cfg, L, N, k, want_outputs, fill):
    dev = "cuda"
    out = dict(load=torch.full((L, cfg.P), fill, dtype=torch.int64, device=dev),
               comm_span=torch.full((L, cfg.F), fill, dtype=torch.int64, device=dev),
               comm_remote=torch.full((L, cfg.F), fill, dtype=torch.int64, device=dev),
               ntok=torch.full((cfg.F,), fill, dtype=torch.int64, device=dev),
               fairness=torch.full((L + 1, 3), float(fill), dtype=torch.float32, device=dev))
    if want_outputs:
        out["cost"] = torch.full((L, N), 255, dtype=torch.uint8, device=dev)
        out["serve"] = torch.full((L, N, k), 99, dtype=torch.int8, device=dev)
    return out


def _compare(tacg, ctx, case, offset, rho):
    cfg, idx, fam, primary, want_outputs = case
    L, N, k = idx.shape
    st_ref = torch.linspace(0.0, 5.0, L * cfg.P, dtype=torch.float64, device="cuda").reshape(L, cfg.P).contiguous()
    st_new = st_ref.clone()
    ref = tacg.tacg_eval_placement(ctx, idx, fam, cfg.E, cfg.F, cfg.P, primary, None, rho=rho, token_offset=offset,
                                   load_state=st_ref, want_cost=want_outputs, want_serve=want_outputs)
    out = _outputs(cfg, L, N, k, want_outputs, fill=-7)
    tacg.tacg_eval_primary_noalloc(ctx, idx, fam, cfg.E, cfg.F, cfg.P, primary, out, rho=rho, token_offset=offset,
                                   load_state=st_new)
    torch.cuda.synchronize()
    for key in ("load", "comm_span", "comm_remote", "ntok"):
        assert torch.equal(out[key], ref[key]), key
    if want_outputs:
        assert torch.equal(out["cost"], ref["cost"])
        assert torch.equal(out["serve"], ref["serve"])
    assert (st_new.cpu().numpy().view(np.uint64) == st_ref.cpu().numpy().view(np.uint64)).all()
    assert np.allclose(out["fairness"].cpu().numpy(), ref["fairness"].cpu().numpy(), rtol=1e-5, atol=1e-7)
    assert int(out["ntok"].sum()) > 0 and int(out["load"].sum()) > 0        # not two empty results


def test_no_alloc_entry_matches_the_existing_path_twice_in_a_row(tacg, ctx):
    ctx.check(ctx.tacg_eval_primary_noalloc_prepare(), "prepare")
    first = _case(3, 70001, 3, seed=21, want_outputs=True)       # k = 8, P = 16, ragged last slice
    second = _case(2, 300000, 2, seed=22, want_outputs=False)    # k = 6, P = 8, other row width, more items
    third = _case(1, 4096, 1, seed=23, want_outputs=True)        # k = 2: the smallest rows over the leftovers
    _compare(tacg, ctx, first, offset=0, rho=0.995)
    _compare(tacg, ctx, second, offset=5, rho=0.9)
    _compare(tacg, ctx, third, offset=1, rho=0.5)
    _compare(tacg, ctx, first, offset=3, rho=0.995)


def test_no_alloc_entry_leaves_the_allocator_alone(tacg, ctx):
    case = _case(3, 50000, 2, seed=24, want_outputs=False)
    cfg, idx, fam, primary, _ = case
    L, N, k = idx.shape
    out = _outputs(cfg, L, N, k, False, fill=0)
    tacg.tacg_eval_primary_noalloc(ctx, idx, fam, cfg.E, cfg.F, cfg.P, primary, out)      # first use on the device
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    torch0 = torch.cuda.memory_allocated()
    for _ in range(3):
        tacg.tacg_eval_primary_noalloc(ctx, idx, fam, cfg.E, cfg.F, cfg.P, primary, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0 and torch.cuda.memory_allocated() == torch0


def test_no_alloc_entry_refuses_what_does_not_fit(tacg, ctx):
    # rows: L * ceil(N / slice) * align4(P + 3F + 2) words, slice <= 32768.  P = 64, F = 8 -> 92 words; 256 layers x 128 slices
    L, N, k, E, F, P = 256, 128 * 32768, 1, 64, 8, 64
    assert L * (N // 32768) * 92 * 4 > tacg.NOALLOC_SCRATCH_BYTES
    idx = torch.zeros((L, N, k), dtype=torch.int16, device="cuda")
    fam = torch.zeros((N,), dtype=torch.int8, device="cuda")
    primary = torch.zeros((L, E), dtype=torch.int8, device="cuda")
    out = dict(load=torch.empty((L, P), dtype=torch.int64, device="cuda"),
               comm_span=torch.empty((L, F), dtype=torch.int64, device="cuda"),
               comm_remote=torch.empty((L, F), dtype=torch.int64, device="cuda"),
               ntok=torch.empty((F,), dtype=torch.int64, device="cuda"),
               fairness=torch.empty((L + 1, 3), dtype=torch.float32, device="cuda"))
    with pytest.raises(tacg.TacgError) as err:
        tacg.tacg_eval_primary_noalloc(ctx, idx, fam, E, F, P, primary, out)
    assert err.value.code == -2 and "fixed array" in str(err.value)
    # the context still works after the refusal
    ok = tacg.tacg_eval_placement(ctx, idx[:2].contiguous(), fam, E, F, P, primary[:2].contiguous())
    torch.cuda.synchronize()
    assert int(ok["ntok"].sum()) == N

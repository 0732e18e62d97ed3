"""The evaluator's launch modes against the C oracle, element by element (integers bit-exact, EMA bits, fairness 1e-5):

  * replicas with ONE micro-batch over a long trace (microbatch = 0 and N >> 512): the case in which round 1's kernel
    met at a grid barrier without a cooperative launch;
  * the literal per-token Eq. 15, microbatch = 1, on a long trace: one warp per layer, and the
    library's scratch must not grow with the number of micro-batches (round 1 reserved L*nmb*P*8 bytes);
  * short micro-batches on both sides of the switch between the one-warp kernel and the scan + chain kernels;
  * few layers with long micro-batches: the chain kernel's cooperative grid mode;
  * shapes outside the record format of the scan kernel, which the chain kernel serves from the trace: odd k, more than
    15 replicated experts in a layer, P > 32 (64-bit partition sets), every expert replicated.
"""
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


def _u64(t):
    return t.cpu().numpy().view(np.uint64)


def _check(tacg, ctx, E, F, P, idx, fam, primary, replicas, theta, rho, B, offset=0, outputs=True):
    L = idx.shape[0]
    want = cbind.eval_placement(idx.numpy(), fam.numpy(), E, F, P, primary, replicas, theta=theta, rho=rho, microbatch=B,
                                token_offset=offset, want_cost=outputs, want_serve=outputs, load_state=np.zeros((L, P)))
    st = torch.zeros((L, P), dtype=torch.float64, device="cuda")
    got = tacg.tacg_eval_placement(ctx, idx.cuda(), fam.cuda(), E, F, P, torch.from_numpy(primary).cuda(),
                                   None if replicas is None else torch.from_numpy(replicas).cuda(), theta=theta, rho=rho,
                                   microbatch=B, token_offset=offset, load_state=st, want_cost=outputs, want_serve=outputs)
    torch.cuda.synchronize()
    assert (_u64(got["load"]) == want["load"]).all()
    assert (_u64(got["comm_span"]) == want["comm_span"]).all()
    assert (_u64(got["comm_remote"]) == want["comm_remote"]).all()
    assert (_u64(got["ntok"]) == want["ntok"]).all()
    if outputs:
        assert (got["cost"].cpu().numpy() == want["cost"]).all()
        assert (got["serve"].cpu().numpy() == want["serve"]).all()
    assert (st.cpu().numpy().view(np.uint64) == want["load_state"].view(np.uint64)).all()
    assert np.allclose(got["fairness"].cpu().numpy().astype(np.float64), want["fairness"], rtol=1e-5, atol=1e-7)
    return got


def _trace(cfg_id, N, L):
    cfg = tracegen.scaled(tracegen.get_config(cfg_id), N=N, N_eval=N, L=L)
    idx, fam = tracegen.gen_trace(cfg, tracegen.make_params(cfg), eval_trace=True)
    return cfg, idx, fam


@pytest.mark.parametrize("cfg_id,N,L", [(3, 300000, 2), (5, 200003, 1)])
def test_replicas_single_microbatch_long_trace(tacg, ctx, cfg_id, N, L):
    cfg, idx, fam = _trace(cfg_id, N, L)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, L, seed=5)
    replicas = tracegen.random_replicas(primary, cfg.P, cfg.r, cfg.n_rep, seed=6)
    _check(tacg, ctx, cfg.E, cfg.F, cfg.P, idx, fam, primary, replicas, 0.15, 0.995, 0)
    _check(tacg, ctx, cfg.E, cfg.F, cfg.P, idx, fam, primary, replicas, 0.15, 0.995, N + 7, outputs=False)


@pytest.mark.parametrize("cfg_id,N,L", [(3, 150000, 3), (5, 120001, 1)])
def test_literal_per_token_ema_long_trace(tacg, ctx, cfg_id, N, L):
    cfg, idx, fam = _trace(cfg_id, N, L)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, L, seed=7)
    replicas = tracegen.random_replicas(primary, cfg.P, cfg.r, cfg.n_rep, seed=8)
    torch.cuda.synchronize()
    before = torch.cuda.mem_get_info()[0]
    _check(tacg, ctx, cfg.E, cfg.F, cfg.P, idx, fam, primary, replicas, 0.15, 0.995, 1, offset=3)
    # the call itself holds inputs and outputs (a few MB); scratch per micro-batch would be hundreds of MB here
    assert before - torch.cuda.mem_get_info()[0] < 256 * 1024 * 1024


@pytest.mark.parametrize("cfg_id,N,L,B,offset", [(5, 300007, 1, 65536, 0), (3, 200000, 3, 40000, 5), (5, 150000, 4, 32768, 1),
                                                  (4, 140000, 2, 65536, 9)])
def test_few_layers_long_microbatches(tacg, ctx, cfg_id, N, L, B, offset):
    """L <= 4 with micro-batches of 32 K tokens or more: more CTAs per layer than a cluster holds (cooperative launch,
    counts exchanged through global memory), several micro-batches and a ragged last one."""
    cfg, idx, fam = _trace(cfg_id, N, L)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, L, seed=15)
    replicas = tracegen.random_replicas(primary, cfg.P, cfg.r, cfg.n_rep, seed=16)
    _check(tacg, ctx, cfg.E, cfg.F, cfg.P, idx, fam, primary, replicas, 0.15, 0.995, B, offset=offset)
    _check(tacg, ctx, cfg.E, cfg.F, cfg.P, idx, fam, primary, replicas, 0.05, 0.9, B, offset=offset, outputs=False)


@pytest.mark.parametrize("B", [2, 31, 33, 512, 1023, 1024, 1025, 3000, 8192, 8193, 20000])
def test_microbatch_lengths_around_the_kernel_switch(tacg, ctx, B):
    cfg, idx, fam = _trace(3, 50021, 2)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, 2, seed=9)
    replicas = tracegen.random_replicas(primary, cfg.P, cfg.r, 6, seed=10)
    _check(tacg, ctx, cfg.E, cfg.F, cfg.P, idx, fam, primary, replicas, 0.1, 0.9, B, offset=11)


@pytest.mark.parametrize("cfg_id,N,L,B", [(3, 70000, 2, 8192), (5, 140000, 1, 65536), (4, 60000, 3, 4096)])
def test_initial_state_with_ties_and_signed_zeros(tacg, ctx, cfg_id, N, L, B):
    """The chain kernel orders an expert's candidates by integer keys of the loads (order_key): equal loads must keep
    slot order, +0.0 and -0.0 are equal, and a guard decided on the very first micro-batch has to see the given state.
    Rounded initial loads give many exact ties; the three launch modes of the chain kernel each get a case."""
    cfg, idx, fam = _trace(cfg_id, N, L)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, L, seed=31)
    replicas = tracegen.random_replicas(primary, cfg.P, cfg.r, cfg.n_rep, seed=32)
    rng = np.random.default_rng(33)
    state0 = np.round(rng.uniform(0.0, 3.0, size=(L, cfg.P))) * 1000.0        # few distinct values: ties
    state0[:, ::5] = -0.0
    state0[:, 1::7] = 0.0
    want = cbind.eval_placement(idx.numpy(), fam.numpy(), cfg.E, cfg.F, cfg.P, primary, replicas, theta=0.15, rho=0.995,
                                microbatch=B, load_state=state0.copy())
    st = torch.from_numpy(state0.copy()).cuda()
    got = tacg.tacg_eval_placement(ctx, idx.cuda(), fam.cuda(), cfg.E, cfg.F, cfg.P, torch.from_numpy(primary).cuda(),
                                   torch.from_numpy(replicas).cuda(), theta=0.15, rho=0.995, microbatch=B, load_state=st)
    torch.cuda.synchronize()
    assert (_u64(got["load"]) == want["load"]).all()
    assert (_u64(got["comm_span"]) == want["comm_span"]).all()
    assert (_u64(got["comm_remote"]) == want["comm_remote"]).all()
    assert (st.cpu().numpy().view(np.uint64) == want["load_state"].view(np.uint64)).all()


def _random_trace(E, k, L, N, F, seed):
    g = torch.Generator().manual_seed(seed)
    idx = torch.stack([torch.stack([torch.randperm(E, generator=g)[:k] for _ in range(N)]) for _ in range(L)]).to(torch.int16)
    fam = torch.randint(0, F, (N,), generator=g).to(torch.int8)
    return idx, fam


@pytest.mark.parametrize("E,k,P,cap,r,n_rep,B", [
    (40, 5, 8, 5, 2, 6, 2000),        # odd k: no packed loads, no records
    (64, 8, 8, 8, 2, 30, 2048),       # more replicated experts than the 4-bit rank fields name
    (64, 8, 8, 8, 3, 64, 1500),       # every expert replicated
    (128, 6, 48, 3, 4, 10, 2048),     # P > 32: 64-bit partition sets; r = 4: five candidates per expert
    (96, 4, 64, 2, 8, 12, 4096),      # the ABI's limits of P and r
])
def test_shapes_outside_the_record_format(tacg, ctx, E, k, P, cap, r, n_rep, B):
    L, N, F = 2, 9000, 3
    idx, fam = _random_trace(E, k, L, N, F, seed=E + k)
    idx[0, 17, 0] = -1                       # an empty slot
    fam[23] = -1                             # a padding token
    primary = tracegen.random_placement(E, P, cap, L, seed=12)
    replicas = tracegen.random_replicas(primary, P, r, n_rep, seed=13)
    _check(tacg, ctx, E, F, P, idx, fam, primary, replicas, 0.2, 0.97, B, offset=1)


def test_binding_refuses_short_buffers_and_foreign_streams(tacg, ctx):
    """a family tensor shorter than N, or a primary / replicas tensor whose size does not match [L,E] /
    [L,E,r], would be an out-of-bounds device read; a context used under another stream would race silently."""
    cfg, idx, fam = _trace(3, 4096, 2)
    primary = torch.from_numpy(tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, 2, seed=1)).cuda()
    replicas = torch.from_numpy(tracegen.random_replicas(primary.cpu().numpy(), cfg.P, 2, 4, seed=2)).cuda()
    with pytest.raises(ValueError):
        tacg.tacg_eval_placement(ctx, idx.cuda(), fam[:100].cuda(), cfg.E, cfg.F, cfg.P, primary, replicas)
    with pytest.raises(ValueError):
        tacg.tacg_eval_placement(ctx, idx.cuda(), fam.cuda(), cfg.E, cfg.F, cfg.P, primary[:1].contiguous(), replicas)
    with pytest.raises(ValueError):
        tacg.tacg_eval_placement(ctx, idx.cuda(), fam.cuda(), cfg.E, cfg.F, cfg.P, primary, replicas[:, :64].contiguous())
    with pytest.raises(ValueError):
        tacg.tacg_coact_accumulate(ctx, idx.cuda(), fam[:7].cuda(), cfg.E, cfg.F)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        with pytest.raises(ValueError):
            tacg.tacg_coact_accumulate(ctx, idx.cuda(), fam.cuda(), cfg.E, cfg.F)
        with tacg.Context(0, side) as c2:                       # a context of its own for the other stream works
            out = tacg.tacg_coact_accumulate(c2, idx.cuda(), fam.cuda(), cfg.E, cfg.F)
            side.synchronize()
            assert int(out["ntok"].sum()) == 4096

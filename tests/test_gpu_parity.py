"""Parity of the CUDA path (through the C-ABI, via the ctypes binding) against the oracle,
element by element, on the same seeded inputs.  Integers bit-exact; fp32 outputs within the
tolerances of DESIGN.md "Tolerances" (1e-5 relative)."""
import numpy as np
import pytest
import torch

import tracegen
from oracle import cbind, ref

pytestmark = pytest.mark.gpu

F32 = np.float32


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


def _trace(cfg_id, N, L=None, seed=None, eval_trace=False):
    cfg = tracegen.get_config(cfg_id)
    cfg = tracegen.scaled(cfg, N=N, N_eval=N, L=min(cfg.L, L or cfg.L))
    params = tracegen.make_params(cfg)
    idx, fam = tracegen.gen_trace(cfg, params, seed=seed, eval_trace=eval_trace)
    return cfg, idx, fam


def _u32(t):
    return t.cpu().numpy().view(np.uint32)


def _u64(t):
    return t.cpu().numpy().view(np.uint64)


# --------------------------------------------------------------------------- S1 + S2
COACT_CASES = [
    # cfg, N, L  -- sizes span several CTAs and a ragged tail (N not a multiple of any tile)
    (1, 4096, 1), (1, 37, 1), (2, 20011, 3), (3, 9973, 2), (4, 6007, 2), (5, 12345, 1),
]


PATH_FLAG = {"hist": 0x10, "auto": 0x00, "mma": 0x20}


@pytest.mark.parametrize("path", ["hist", "auto", "mma"])
@pytest.mark.parametrize("cfg_id,N,L", COACT_CASES)
def test_coact_counts_bit_exact(tacg, ctx, cfg_id, N, L, path):
    cfg, idx, fam = _trace(cfg_id, N, L)
    D, C, ntok = cbind.coact(idx.numpy(), fam.numpy(), cfg.E, cfg.F)
    flags = tacg.TACG_ZERO_FIRST | PATH_FLAG[path]
    out = tacg.tacg_coact_accumulate(ctx, idx.cuda(), fam.cuda(), cfg.E, cfg.F, flags=flags)
    torch.cuda.synchronize()
    assert (_u32(out["D"]) == D).all()
    assert (_u32(out["C"]) == C).all()
    assert (_u64(out["ntok"]) == ntok).all()
    # accumulate semantics: a second call without ZERO_FIRST doubles everything
    out2 = tacg.tacg_coact_accumulate(ctx, idx.cuda(), fam.cuda(), cfg.E, cfg.F, D=out["D"], Cm=out["C"],
                                      ntok=out["ntok"], flags=flags & ~tacg.TACG_ZERO_FIRST)
    torch.cuda.synchronize()
    assert (_u32(out2["D"]) == 2 * D).all() and (_u32(out2["C"]) == 2 * C).all()
    assert (_u64(out2["ntok"]) == 2 * ntok).all()


@pytest.mark.parametrize("path", ["hist", "auto", "mma"])
def test_coact_skip_rules_and_generic_k(tacg, ctx, path):
    """Negative ids = empty slots, negative family = padding; odd k and unaligned views use the generic loader."""
    rng = np.random.default_rng(5)
    for (E, k, F, N, L) in [(16, 3, 3, 1000, 2), (64, 6, 4, 3001, 2), (128, 8, 4, 2500, 1), (40, 5, 1, 777, 1)]:
        idx = np.stack([np.stack([rng.permutation(E)[:k] for _ in range(N)]) for _ in range(L)]).astype(np.int16)
        idx[rng.random(idx.shape) < 0.1] = -1
        fam = rng.integers(0, F, size=N).astype(np.int8)
        fam[rng.random(N) < 0.05] = -1
        if path == "mma" and k % 2:
            continue                                    # tcgen05 path: even k only (vector row loads)
        D, C, ntok = cbind.coact(idx, fam, E, F)
        flags = tacg.TACG_ZERO_FIRST | PATH_FLAG[path]
        out = tacg.tacg_coact_accumulate(ctx, torch.from_numpy(idx).cuda(), torch.from_numpy(fam).cuda(), E, F,
                                         flags=flags)
        torch.cuda.synchronize()
        assert (_u32(out["D"]) == D).all() and (_u32(out["C"]) == C).all() and (_u64(out["ntok"]) == ntok).all()


def test_coact_handworked(tacg, ctx, golden_trace):
    g = golden_trace
    fam = torch.tensor(g["family"][0], dtype=torch.int8).cuda()
    idx = torch.tensor(g["experts"], dtype=torch.int16)[None].contiguous().cuda()
    out = tacg.tacg_coact_accumulate(ctx, idx, fam, 4, 2)
    D = _u32(out["D"])
    assert D[0, 0].tolist() == g["D0"][0] and D[0, 1].tolist() == g["D1"][0]
    C = _u32(out["C"])
    want = np.zeros((2, 4, 4), dtype=np.uint32)
    for f, i, j, c in g["C"]:
        want[int(f), int(i), int(j)] = want[int(f), int(j), int(i)] = int(c)
    assert (C[0] == want).all()


def test_coact_empty_and_errors(tacg, ctx):
    dev = "cuda"
    idx = torch.empty((2, 0, 6), dtype=torch.int16, device=dev)
    fam = torch.empty((0,), dtype=torch.int8, device=dev)
    out = tacg.tacg_coact_accumulate(ctx, idx, fam, 64, 4)
    torch.cuda.synchronize()
    assert int(out["D"].abs().sum()) == 0 and int(out["C"].abs().sum()) == 0
    idx = torch.zeros((1, 8, 2), dtype=torch.int16, device=dev)
    fam = torch.zeros((8,), dtype=torch.int8, device=dev)
    D = torch.zeros((1, 1, 4), dtype=torch.int32, device=dev)
    Cm = torch.zeros((1, 1, 4, 4), dtype=torch.int32, device=dev)
    nt = torch.zeros((1,), dtype=torch.int64, device=dev)
    assert ctx.tacg_coact_accumulate(idx, fam, 8, 2, 1, 4, 1, None, Cm, nt, 0) == -1          # NULL
    assert ctx.tacg_coact_accumulate(idx, fam, 8, 17, 1, 4, 1, D, Cm, nt, 0) == -2            # k > 16
    assert ctx.tacg_coact_accumulate(idx, fam, 8, 2, 1, 513, 1, D, Cm, nt, 0) == -2           # E > 512
    assert ctx.tacg_coact_accumulate(idx, fam, 8, 2, 1, 4, 9, D, Cm, nt, 0) == -2             # F > 8
    # validation: duplicate expert inside a token (both slots are 0)
    assert ctx.tacg_coact_accumulate(idx, fam, 8, 2, 1, 4, 1, D, Cm, nt, tacg.TACG_VALIDATE) == -3
    assert int(D.sum()) == 0 and int(Cm.sum()) == 0, "a failed call must not write outputs"
    idx2 = torch.tensor([[[0, 1], [2, 9]]], dtype=torch.int16, device=dev)
    assert ctx.tacg_coact_accumulate(idx2, fam[:2].contiguous(), 2, 2, 1, 4, 1, D, Cm, nt, tacg.TACG_VALIDATE) == -3
    assert "record 1" in ctx.detail()
    # the tensor path refuses what it cannot do (odd k, E > 256) before touching the outputs
    big = torch.zeros((1, 8, 2), dtype=torch.int16, device=dev)
    Db = torch.zeros((1, 1, 300), dtype=torch.int32, device=dev)
    Cb = torch.zeros((1, 1, 300, 300), dtype=torch.int32, device=dev)
    assert ctx.tacg_coact_accumulate(big, fam, 8, 2, 1, 300, 1, Db, Cb, nt, tacg.TACG_PATH_MMA) == -2
    odd = torch.zeros((1, 8, 3), dtype=torch.int16, device=dev)
    assert ctx.tacg_coact_accumulate(odd, fam, 8, 3, 1, 4, 1, D, Cm, nt, tacg.TACG_PATH_MMA) == -2
    assert ctx.tacg_coact_accumulate(idx, fam, 8, 2, 1, 4, 1, D, Cm, nt,
                                     tacg.TACG_PATH_MMA | tacg.TACG_PATH_HIST) == -2          # both paths forced
    idx3 = torch.tensor([[[0, 1], [2, 3]]], dtype=torch.int16, device=dev)
    assert ctx.tacg_coact_accumulate(idx3, fam[:2].contiguous(), 2, 2, 1, 4, 1, D, Cm, nt, tacg.TACG_VALIDATE) == 0


# --------------------------------------------------------------------------- S3..S7
def _tol_check(got, want, name):
    got = np.asarray(got, dtype=np.float64)
    err = np.abs(got - want)
    bound = 1e-5 * np.maximum(np.abs(want), 1e-6)
    bad = err > bound
    assert not bad.any(), f"{name}: max err {err.max():.3e}, {bad.sum()} entries over 1e-5 relative"


@pytest.mark.parametrize("cfg_id,N,L", [(1, 4096, 1), (2, 30000, 3), (3, 20000, 2), (4, 20000, 2), (5, 50000, 1)])
@pytest.mark.parametrize("alpha,tau", [(0.25, 1.0), (0.0, 1.0), (0.7, 0.5)])
def test_affinity_swapgain_parity(tacg, ctx, cfg_id, N, L, alpha, tau):
    cfg, idx, fam = _trace(cfg_id, N, L)
    D, C, ntok = cbind.coact(idx.numpy(), fam.numpy(), cfg.E, cfg.F)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, cfg.L, seed=11)
    a32, t32, e32 = float(F32(alpha)), float(F32(tau)), float(F32(1e-6))     # the ABI takes floats
    want = cbind.affinity_swapgain(D, C, ntok, cfg.P, primary, alpha=a32, tau=t32, eps=e32)
    dD = torch.from_numpy(D.view(np.int32)).cuda()
    dC = torch.from_numpy(C.view(np.int32)).cuda()
    dn = torch.from_numpy(ntok.view(np.int64)).cuda()
    got = tacg.tacg_affinity_swapgain(ctx, dD, dC, dn, cfg.P, cfg.capacity, torch.from_numpy(primary).cuda(),
                                      alpha=alpha, tau=tau, eps=1e-6)
    torch.cuda.synchronize()
    _tol_check(got["pref"].cpu().numpy(), want["pref"], "pref")
    _tol_check(got["W"].cpu().numpy(), want["W"], "W")
    _tol_check(got["aff"].cpu().numpy(), want["aff"], "aff")
    # G: 1e-5 relative to the operand magnitude (Q14)
    aff, W = want["aff"], want["W"]
    G = got["gain"].cpu().numpy().astype(np.float64)
    for l in range(cfg.L):
        pr = primary[l].astype(np.int64)
        ia = aff[l][np.arange(cfg.E), pr]                      # aff[i, a]
        ib = aff[l][:, pr]                                     # aff[i, b(j)]
        mag = np.abs(ib) + np.abs(ib.T) + np.abs(ia)[:, None] + np.abs(ia)[None, :] + 2 * np.abs(W[l])
        err = np.abs(G[l] - want["gain"][l])
        assert (err <= 1e-5 * np.maximum(mag, 1e-6)).all(), f"gain layer {l}: max err {err.max():.3e}"
        assert (G[l][pr[:, None] == pr[None, :]] == 0).all()


def test_affinity_handworked(tacg, ctx, golden_trace):
    g = golden_trace
    fam = torch.tensor(g["family"][0], dtype=torch.int8).cuda()
    idx = torch.tensor(g["experts"], dtype=torch.int16)[None].contiguous().cuda()
    co = tacg.tacg_coact_accumulate(ctx, idx, fam, 4, 2)
    primary = torch.tensor(g["primary"], dtype=torch.int8).cuda()
    out = tacg.tacg_affinity_swapgain(ctx, co["D"], co["C"], co["ntok"], 2, 2, primary, alpha=0.25, tau=1.0, eps=1e-6)
    assert np.allclose(out["pref"][0].cpu().numpy(), np.array(g["pref"]), atol=1.5e-6)
    assert np.allclose(out["W"][0].cpu().numpy(), np.array(g["W"]), atol=1.5e-6)
    assert np.allclose(out["aff"][0].cpu().numpy(), np.array(g["aff"]), atol=1.5e-6)
    G = np.zeros((4, 4))
    for i, j, v in g["G"]:
        G[int(i), int(j)] = G[int(j), int(i)] = v
    assert np.allclose(out["gain"][0].cpu().numpy(), G, atol=3e-6)


def test_affinity_optional_outputs_and_errors(tacg, ctx):
    cfg, idx, fam = _trace(1, 512, 1)
    co = tacg.tacg_coact_accumulate(ctx, idx.cuda(), fam.cuda(), cfg.E, cfg.F)
    out = tacg.tacg_affinity_swapgain(ctx, co["D"], co["C"], co["ntok"], cfg.P, cfg.capacity, None, want=("pref", "W"))
    assert out["aff"] is None and out["gain"] is None and out["W"] is not None
    pr = torch.zeros((1, cfg.E), dtype=torch.int8, device="cuda")
    W = torch.empty((1, cfg.E, cfg.E), dtype=torch.float32, device="cuda")
    # E > P*capacity
    assert ctx.tacg_affinity_swapgain(co["D"], co["C"], co["ntok"], 1, cfg.E, cfg.F, 2, 2, pr, 0.25, 1.0, 1e-6,
                                      None, W, None, None) == -2
    # aff requested without primary
    aff = torch.empty((1, cfg.E, cfg.P), dtype=torch.float32, device="cuda")
    assert ctx.tacg_affinity_swapgain(co["D"], co["C"], co["ntok"], 1, cfg.E, cfg.F, cfg.P, cfg.capacity, None,
                                      0.25, 1.0, 1e-6, None, None, aff, None) == -1


# --------------------------------------------------------------------------- S8..S12
def _eval_both(tacg, ctx, cfg, idx, fam, primary, replicas, theta, rho, B, offset=0, state0=None):
    want = cbind.eval_placement(idx.numpy(), fam.numpy(), cfg.E, cfg.F, cfg.P, primary, replicas, theta=theta, rho=rho,
                                microbatch=B, token_offset=offset, want_cost=True, want_serve=True,
                                load_state=np.zeros((cfg.L, cfg.P)) if state0 is None else state0.copy())
    st = torch.zeros((cfg.L, cfg.P), dtype=torch.float64, device="cuda") if state0 is None \
        else torch.from_numpy(state0.copy()).cuda()
    got = tacg.tacg_eval_placement(ctx, idx.cuda(), fam.cuda(), cfg.E, cfg.F, cfg.P, torch.from_numpy(primary).cuda(),
                                   None if replicas is None else torch.from_numpy(replicas).cuda(), theta=theta,
                                   rho=rho, microbatch=B, token_offset=offset, load_state=st, want_cost=True,
                                   want_serve=True)
    torch.cuda.synchronize()
    return want, got


def _assert_eval_equal(want, got):
    assert (_u64(got["load"]) == want["load"]).all()
    assert (_u64(got["comm_span"]) == want["comm_span"]).all()
    assert (_u64(got["comm_remote"]) == want["comm_remote"]).all()
    assert (_u64(got["ntok"]) == want["ntok"]).all()
    assert (got["cost"].cpu().numpy() == want["cost"]).all()
    assert (got["serve"].cpu().numpy() == want["serve"]).all()
    # EMA state: bit-exact doubles (Q19)
    assert (got["load_state"].cpu().numpy().view(np.uint64) == want["load_state"].view(np.uint64)).all()
    fair = got["fairness"].cpu().numpy().astype(np.float64)
    assert np.allclose(fair, want["fairness"], rtol=1e-5, atol=1e-7)


@pytest.mark.parametrize("cfg_id,N,L", [(1, 4096, 1), (2, 20011, 3), (3, 9973, 2), (4, 6007, 3), (5, 30001, 1)])
def test_eval_no_replicas(tacg, ctx, cfg_id, N, L):
    cfg, idx, fam = _trace(cfg_id, N, L, eval_trace=True)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, cfg.L, seed=21)
    want, got = _eval_both(tacg, ctx, cfg, idx, fam, primary, None, 0.15, 0.995, 0, offset=5)
    _assert_eval_equal(want, got)
    L_, P_ = want["load"].shape
    assert (want["load"].sum(axis=1) == N * cfg.k).all()
    jain = got["fairness"][:, 0].cpu().numpy()
    assert ((jain >= 1.0 / P_ - 1e-6) & (jain <= 1.0 + 1e-6)).all()


@pytest.mark.parametrize("cfg_id,N,L,r,B", [
    (1, 4096, 1, 1, 256), (3, 40000, 2, 2, 4096), (4, 30011, 3, 2, 5000), (5, 100003, 1, 3, 8192),
    (3, 5000, 48, 2, 700),      # more layers than fit one CTA group each
    (5, 3000, 1, 3, 1),         # micro-batch of one token: the literal per-token chain
])
@pytest.mark.parametrize("theta,rho", [(0.15, 0.995), (0.0, 0.5), (float("inf"), 1.0)])
def test_eval_gesr(tacg, ctx, cfg_id, N, L, r, B, theta, rho):
    cfg, idx, fam = _trace(cfg_id, N, L, eval_trace=True)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, cfg.L, seed=31)
    replicas = tracegen.random_replicas(primary, cfg.P, r, max(4, cfg.n_rep * 2), seed=32)
    rng = np.random.default_rng(33)
    state0 = rng.random((cfg.L, cfg.P)) * 50.0
    want, got = _eval_both(tacg, ctx, cfg, idx, fam, primary, replicas, theta, rho, B, offset=7, state0=state0)
    _assert_eval_equal(want, got)


def test_eval_handworked(tacg, ctx, golden_trace):
    g = golden_trace
    fam = torch.tensor(g["family"][0], dtype=torch.int8).cuda()
    idx = torch.tensor(g["experts"], dtype=torch.int16)[None].contiguous().cuda()
    primary = torch.tensor(g["primary"], dtype=torch.int8).cuda()
    out = tacg.tacg_eval_placement(ctx, idx, fam, 4, 2, 2, primary)
    assert _u64(out["load"])[0].tolist() == g["load"][0]
    assert _u64(out["comm_span"])[0].tolist() == g["comm_span"][0]
    assert _u64(out["comm_remote"])[0].tolist() == g["comm_remote"][0]
    fair = out["fairness"].cpu().numpy()
    assert abs(fair[0, 0] - g["jain"][0][0]) < 1.5e-6 and abs(fair[0, 1] - g["maxvio"][0][0]) < 1.5e-6
    rep = torch.tensor(g["gesr_replicas"], dtype=torch.int8)[None].contiguous().cuda()
    st = torch.zeros((1, 2), dtype=torch.float64, device="cuda")
    out = tacg.tacg_eval_placement(ctx, idx, fam, 4, 2, 2, primary, rep, theta=0.15, rho=0.995, microbatch=4,
                                   load_state=st, want_serve=True)
    assert out["serve"][0].cpu().numpy().tolist() == [[int(x) for x in row] for row in g["gesr_serve"]]
    assert _u64(out["load"])[0].tolist() == g["gesr_load"][0]
    assert np.allclose(st.cpu().numpy()[0], g["gesr_state_final"][0], atol=1e-12)
    assert int(_u64(out["comm_span"]).sum()) == g["gesr_comm_span_total"][0][0]
    assert int(_u64(out["comm_remote"]).sum()) == g["gesr_comm_remote_total"][0][0]


@pytest.mark.parametrize("cfg_id,N,L,r", [(1, 1000, 1, 1), (3, 20000, 2, 2), (5, 50001, 1, 3), (2, 5000, 2, 0)])
def test_gesr_select(tacg, ctx, cfg_id, N, L, r):
    cfg, idx, fam = _trace(cfg_id, N, L, eval_trace=True)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, cfg.L, seed=41)
    replicas = tracegen.random_replicas(primary, cfg.P, r, max(4, cfg.n_rep * 2), seed=42) if r else None
    rng = np.random.default_rng(43)
    for theta, scale in ((0.15, 100.0), (0.0, 1.0), (float("inf"), 10.0), (0.15, 0.0)):
        snap = rng.random((cfg.L, cfg.P)) * scale
        want = cbind.gesr_select(idx.numpy(), cfg.E, cfg.P, primary, replicas, snap, theta, token_offset=13)
        got = tacg.gesr_select(ctx, idx.cuda(), cfg.E, cfg.P, torch.from_numpy(primary).cuda(),
                               None if replicas is None else torch.from_numpy(replicas).cuda(),
                               torch.from_numpy(snap).cuda(), theta, token_offset=13)
        torch.cuda.synchronize()
        assert (got.cpu().numpy() == want).all()


def test_gesr_fallback_all_infeasible(tacg, ctx):
    """Every candidate of the replicated expert is over the guard: the full candidate set is used."""
    E, P, k = 8, 4, 2
    primary = np.array([[0, 0, 1, 1, 2, 2, 3, 3]], dtype=np.int8)
    replicas = np.full((1, E, 2), -1, dtype=np.int8)
    replicas[0, 0] = [1, -1]
    snap = np.array([[10.0, 9.0, 0.0, 0.0]])          # mean 4.75, threshold 5.46: partitions 0 and 1 infeasible
    idx = np.array([[[0, 4], [0, 6], [4, 0]]], dtype=np.int16)
    want = cbind.gesr_select(idx, E, P, primary, replicas, snap, 0.15, token_offset=2)
    got = tacg.gesr_select(ctx, torch.from_numpy(idx).cuda(), E, P, torch.from_numpy(primary).cuda(),
                           torch.from_numpy(replicas).cuda(), torch.from_numpy(snap).cuda(), 0.15, token_offset=2)
    assert (got.cpu().numpy() == want).all()
    assert got.cpu().numpy()[0, 0, 0] == 1              # home = 2: neither is local, fallback picks the less loaded of {0,1}


def test_eval_validate_placement(tacg, ctx):
    cfg, idx, fam = _trace(1, 256, 1)
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, 1, seed=1)
    bad = primary.copy()
    bad[0, 3] = cfg.P                                   # out of range
    with pytest.raises(tacg.TacgError) as ei:
        tacg.tacg_eval_placement(ctx, idx.cuda(), fam.cuda(), cfg.E, cfg.F, cfg.P, torch.from_numpy(bad).cuda(),
                                 flags=tacg.TACG_VALIDATE)
    assert ei.value.code == -4
    rep = np.full((1, cfg.E, 1), -1, dtype=np.int8)
    rep[0, 2, 0] = primary[0, 2]                        # replica equal to the primary
    with pytest.raises(tacg.TacgError):
        tacg.tacg_eval_placement(ctx, idx.cuda(), fam.cuda(), cfg.E, cfg.F, cfg.P, torch.from_numpy(primary).cuda(),
                                 torch.from_numpy(rep).cuda(), flags=tacg.TACG_VALIDATE)
    tacg.tacg_eval_placement(ctx, idx.cuda(), fam.cuda(), cfg.E, cfg.F, cfg.P, torch.from_numpy(primary).cuda(),
                             flags=tacg.TACG_VALIDATE)


def test_limits_of_the_abi(tacg, ctx):
    """The largest shapes tacg.h admits (E = 512, P = 64, F = 8, r = 8, k = 16): global-atomic
    co-activation fallback, 64-bit partition masks, generic-k loaders, > 48 KB of shared memory."""
    rng = np.random.default_rng(11)
    E, k, F, P, r, N, L = 512, 16, 8, 64, 8, 3000, 2
    idx = np.stack([np.stack([rng.permutation(E)[:k] for _ in range(N)]) for _ in range(L)]).astype(np.int16)
    idx[rng.random(idx.shape) < 0.05] = -1
    fam = rng.integers(0, F, size=N).astype(np.int8)
    D, C, ntok = cbind.coact(idx, fam, E, F)
    out = tacg.tacg_coact_accumulate(ctx, torch.from_numpy(idx).cuda(), torch.from_numpy(fam).cuda(), E, F,
                                     flags=tacg.TACG_ZERO_FIRST)
    torch.cuda.synchronize()
    assert (_u32(out["D"]) == D).all() and (_u32(out["C"]) == C).all() and (_u64(out["ntok"]) == ntok).all()
    primary = tracegen.random_placement(E, P, 8, L, seed=3)
    replicas = tracegen.random_replicas(primary, P, r, 40, seed=4)
    want = cbind.eval_placement(idx, fam, E, F, P, primary, replicas, theta=0.1, rho=0.9, microbatch=500,
                                token_offset=3, want_cost=True, want_serve=True, load_state=np.zeros((L, P)))
    st = torch.zeros((L, P), dtype=torch.float64, device="cuda")
    got = tacg.tacg_eval_placement(ctx, torch.from_numpy(idx).cuda(), torch.from_numpy(fam).cuda(), E, F, P,
                                   torch.from_numpy(primary).cuda(), torch.from_numpy(replicas).cuda(), theta=0.1,
                                   rho=0.9, microbatch=500, token_offset=3, load_state=st, want_cost=True,
                                   want_serve=True)
    torch.cuda.synchronize()
    got["load_state"] = st
    _assert_eval_equal(want, got)


def test_unaligned_indices_take_the_generic_loaders(tacg, ctx):
    """A trace whose device pointer is not 16-byte aligned (a view one element into a buffer) must give
    the same results through the 2-byte loaders."""
    cfg, idx, fam = _trace(2, 5003, 2)
    flat = torch.empty(idx.numel() + 1, dtype=torch.int16, device="cuda")
    flat[1:] = idx.reshape(-1).cuda()
    view = flat[1:].view(idx.shape)
    assert view.data_ptr() % 16 != 0
    D, C, ntok = cbind.coact(idx.numpy(), fam.numpy(), cfg.E, cfg.F)
    out = tacg.tacg_coact_accumulate(ctx, view, fam.cuda(), cfg.E, cfg.F, flags=tacg.TACG_ZERO_FIRST)
    torch.cuda.synchronize()
    assert (_u32(out["D"]) == D).all() and (_u32(out["C"]) == C).all() and (_u64(out["ntok"]) == ntok).all()
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, cfg.L, seed=5)
    replicas = tracegen.random_replicas(primary, cfg.P, 2, 6, seed=6)
    want = cbind.eval_placement(idx.numpy(), fam.numpy(), cfg.E, cfg.F, cfg.P, primary, replicas, theta=0.15, rho=0.995,
                                microbatch=1000, want_cost=True, want_serve=True, load_state=np.zeros((cfg.L, cfg.P)))
    st = torch.zeros((cfg.L, cfg.P), dtype=torch.float64, device="cuda")
    got = tacg.tacg_eval_placement(ctx, view, fam.cuda(), cfg.E, cfg.F, cfg.P, torch.from_numpy(primary).cuda(),
                                   torch.from_numpy(replicas).cuda(), theta=0.15, rho=0.995, microbatch=1000,
                                   load_state=st, want_cost=True, want_serve=True)
    torch.cuda.synchronize()
    got["load_state"] = st
    _assert_eval_equal(want, got)
    # the tensor path needs aligned rows and says so
    D0 = torch.zeros_like(out["D"]); C0 = torch.zeros_like(out["C"]); n0 = torch.zeros_like(out["ntok"])
    assert ctx.tacg_coact_accumulate(view, fam.cuda(), idx.shape[1], cfg.k, cfg.L, cfg.E, cfg.F, D0, C0, n0,
                                     tacg.TACG_PATH_MMA) == -2

"""The seeded generator produces valid, reproducible traces of the stated shapes.  CPU only."""
import numpy as np
import torch

import tracegen


def test_shapes_distinct_reproducible():
    for cid in (1, 2, 3, 4, 5):
        cfg = tracegen.scaled(tracegen.get_config(cid), N=2000, N_eval=1000, L=2 if cid != 1 and cid != 5 else 1)
        params = tracegen.make_params(cfg)
        idx, fam = tracegen.gen_trace(cfg, params)
        assert idx.shape == (cfg.L, 2000, cfg.k) and idx.dtype == torch.int16
        assert fam.shape == (2000,) and fam.dtype == torch.int8
        a = idx.numpy()
        assert a.min() >= 0 and a.max() < cfg.E
        s = np.sort(a, axis=2)
        assert (s[:, :, 1:] != s[:, :, :-1]).all()          # k distinct experts per token
        assert fam.min() >= 0 and fam.max() < cfg.F
        idx2, fam2 = tracegen.gen_trace(cfg, params)
        assert torch.equal(idx, idx2) and torch.equal(fam, fam2)
        assert tracegen.checksum64(idx) == tracegen.checksum64(idx2)
        eidx, efam = tracegen.gen_trace(cfg, params, eval_trace=True)
        assert eidx.shape == (cfg.L, 1000, cfg.k) and not torch.equal(eidx[:, :1000], idx[:, :1000])
        assert abs(params.pi.sum(-1) - 1).max() < 1e-9


def test_mix_and_generic_mass():
    cfg = tracegen.scaled(tracegen.get_config(5), N=20000, N_eval=20000)
    params = tracegen.make_params(cfg)
    _, fam = tracegen.gen_trace(cfg, params)
    _, efam = tracegen.gen_trace(cfg, params, eval_trace=True)
    h = np.bincount(fam.numpy(), minlength=4) / 20000
    he = np.bincount(efam.numpy(), minlength=4) / 20000
    assert np.allclose(h, cfg.mix, atol=0.02) and np.allclose(he, cfg.mix_eval, atol=0.02)
    g = params.generic[0]
    assert np.allclose(params.pi[0][:, g], 4.0 / cfg.E) and np.allclose(params.pi_eval[0][:, g], 12.0 / cfg.E)


def test_random_placement_feasible():
    pr = tracegen.random_placement(160, 16, 10, 3, seed=1)
    for l in range(3):
        assert np.bincount(pr[l], minlength=16).max() <= 10
    rep = tracegen.random_replicas(pr, 16, 3, 5, seed=2)
    for l in range(3):
        rows = [e for e in range(160) if rep[l, e, 0] >= 0]
        assert len(rows) == 5
        for e in rows:
            v = [x for x in rep[l, e] if x >= 0]
            assert pr[l, e] not in v and len(set(v)) == len(v)


def test_skew_workloads_have_the_stated_shares():
    names = tracegen.skew_workloads(4)
    assert len(names) == 13
    N = 40000
    for w in names:
        fam = tracegen.gen_family_workload(N, w, 4, seed=5)
        assert fam.shape == (N,) and fam.dtype == torch.int8 and fam.min() >= 0 and fam.max() < 4
        assert torch.equal(fam, tracegen.gen_family_workload(N, w, 4, seed=5))
        h = np.bincount(fam.numpy(), minlength=4) / N
        kind, *rest = w.split(":")
        if kind == "balanced":
            assert np.allclose(h, 0.25, atol=0.01)
        elif kind == "single":
            f, s = int(rest[0]), float(rest[1])
            assert abs(h[f] - s) < 0.01 and np.allclose(np.delete(h, f), (1 - s) / 3, atol=0.01)
        elif kind == "phase":
            span = fam.numpy()[: N // 8]
            dom = 0 if rest[0] == "up" else 3
            assert abs((span == dom).mean() - 0.8) < 0.02
        else:
            f = int(rest[0])
            lo = int(0.4 * N)
            assert (fam.numpy()[lo:lo + int(0.15 * N)] == f).all()
            assert abs(h[f] - (0.15 + 0.85 * 0.25)) < 0.01

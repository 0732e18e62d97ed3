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

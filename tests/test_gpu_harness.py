"""the skew sweep of PAPER.md:212-218 / 383 (13 online workloads, one fixed placement each) and
the literal per-token Eq. 15 against the micro-batch snapshot, through paper_2606_01007_b200.harness -- against the same
reports computed with the oracle (integers bit-exact, Comm / Comm. Red. / Jain / MaxVio to 1e-5).

Also pins what the harness adds on the host: the "Frequency" placement (reading Q39) against its definition written out,
and the pooled "Coactivation" placement (tacg_spectral_place on the graph at alpha = 0) against the oracle's
spectral_place on the oracle's own graph.
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


def _setup(tacg, ctx, cfg_id, N, L):
    from paper_2606_01007_b200 import harness
    cfg = tracegen.scaled(tracegen.get_config(cfg_id), N=N, N_eval=N, L=L, microbatch=4096)
    params = tracegen.make_params(cfg)
    bi, bf = tracegen.gen_trace(cfg, params, device="cuda")
    co = tacg.tacg_coact_accumulate(ctx, bi, bf, cfg.E, cfg.F)
    placements = harness.build_placements(ctx, cfg, co["D"], co["C"], co["ntok"])
    return harness, cfg, params, co, placements


def _oracle_row(cfg, idx, fam, primary, replicas, B):
    want = cbind.eval_placement(idx, fam, cfg.E, cfg.F, cfg.P, primary, replicas, theta=0.15, rho=0.995, microbatch=B,
                                load_state=np.zeros((cfg.L, cfg.P)))
    n = int(want["ntok"].sum())
    span = int(want["comm_span"].sum())
    return {"tokens": n, "comm_span_total": span, "comm": span / max(1, n), "jain": float(want["fairness"][-1, 0]),
            "maxvio": float(want["fairness"][-1, 1]), "load": want["load"].astype(np.int64).sum(axis=0).tolist()}


def test_frequency_and_coactivation_placements(tacg, ctx):
    harness, cfg, params, co, placements = _setup(tacg, ctx, 2, 30000, 3)
    D = co["D"].cpu().numpy().view(np.uint32)
    ntok = co["ntok"].cpu().numpy().view(np.uint64)
    # Frequency (Q39): rank by pooled usage, capacity consecutive ranks per partition
    freq = placements["frequency"][0].cpu().numpy()
    for l in range(cfg.L):
        pooled = sum(D[l, f].astype(np.float64) / max(1, int(ntok[f])) for f in range(cfg.F))
        order = sorted(range(cfg.E), key=lambda e: (-pooled[e], e))
        for m in range(cfg.P):
            members = sorted(e for e in range(cfg.E) if freq[l, e] == m)
            assert members == sorted(order[m * cfg.capacity:(m + 1) * cfg.capacity])
        assert np.bincount(freq[l], minlength=cfg.P).max() <= cfg.capacity
    # Coactivation: the oracle's graph at alpha = 0 through the oracle's spectral-then-repair
    C = co["C"].cpu().numpy().view(np.uint32)
    coact = placements["coactivation"][0].cpu().numpy()
    want = cbind.affinity_swapgain(D, C, ntok, cfg.P, np.zeros((cfg.L, cfg.E), dtype=np.int8), alpha=0.0)
    for l in range(cfg.L):
        want_pr, _, _ = ref.spectral_place(want["W"][l].astype(np.float32), cfg.P, cfg.capacity)
        assert coact[l].tolist() == want_pr
    # and it is the task-agnostic graph: no family enters W at alpha = 0
    assert set(placements) >= {"baseline", "frequency", "coactivation", "tacg"}


@pytest.mark.parametrize("cfg_id,N,L", [(2, 20000, 2), (3, 16000, 2)])
def test_skew_report_matches_the_oracle(tacg, ctx, cfg_id, N, L):
    harness, cfg, params, co, placements = _setup(tacg, ctx, cfg_id, N, L)
    seed = cfg.seed + 11
    got = harness.skew_report(ctx, cfg, params, placements, N, seed)
    names = tracegen.skew_workloads(cfg.F)
    assert list(got) == names and len(names) == 13
    for wi, wname in enumerate(names):
        fam = tracegen.gen_family_workload(N, wname, cfg.F, seed + wi, device="cuda")
        idx = tracegen.gen_indices(cfg, params, fam, seed + 100 + wi, eval_trace=True, device="cuda")
        idx_h, fam_h = idx.cpu().numpy(), fam.cpu().numpy()
        base = None
        for name, (pr, rp) in placements.items():
            want = _oracle_row(cfg, idx_h, fam_h, pr.cpu().numpy(), None if rp is None else rp.cpu().numpy(), cfg.microbatch)
            row = got[wname][name]
            assert row["tokens"] == want["tokens"] and row["comm_span_total"] == want["comm_span_total"]
            assert row["load"] == want["load"]
            assert abs(row["jain"] - want["jain"]) <= 1e-5 * abs(want["jain"]) + 1e-7
            assert abs(row["maxvio"] - want["maxvio"]) <= 1e-5 * abs(want["maxvio"]) + 1e-7
            if name == "baseline":
                base = want["comm"]
            red = 100.0 * (base - want["comm"]) / base                      # Eq. 16
            assert abs(row["comm_red_pct"] - red) <= 1e-9 + 1e-9 * abs(red)
    # the placements built from co-activation cut communication on the balanced stream they were calibrated for
    assert got["balanced"]["tacg"]["comm_red_pct"] > 0.0
    assert got["balanced"]["coactivation"]["comm_red_pct"] > 0.0


def test_per_token_gap_matches_the_oracle(tacg, ctx):
    harness, cfg, params, co, placements = _setup(tacg, ctx, 3, 120000, 2)
    ei, ef = tracegen.gen_trace(cfg, params, eval_trace=True, device="cuda")
    pr, rp = placements["tacg+gesr"]
    got = harness.per_token_gap(ctx, cfg, ei, ef, pr, rp)
    lit = _oracle_row(cfg, ei.cpu().numpy(), ef.cpu().numpy(), pr.cpu().numpy(), rp.cpu().numpy(), 1)
    snap = _oracle_row(cfg, ei.cpu().numpy(), ef.cpu().numpy(), pr.cpu().numpy(), rp.cpu().numpy(), cfg.microbatch)
    for key in ("tokens", "comm_span_total", "load"):
        assert got["per_token"][key] == lit[key] and got["microbatch"][key] == snap[key]
    assert abs(got["delta_jain"] - (snap["jain"] - lit["jain"])) <= 1e-6
    assert abs(got["delta_comm_pct"] - 100.0 * (snap["comm"] - lit["comm"]) / lit["comm"]) <= 1e-9

"""Evaluation harness over the library -- consumers of the hot path, not part of it.

  * the placements the paper compares that are derivable from the counts D and C: "Baseline" (the
    default expert order), "Frequency", pooled "Coactivation" (alpha = 0), TACG (alpha = 0.25) and TACG + GESR;
  * the 13 online workloads of the skew sweep (tracegen.skew_workloads) evaluated with one
    fixed placement each, reporting Comm, Comm. Red. (Eq. 16), Jain and MaxVio per workload;
  * the gap between the literal per-token load decay (Eq. 15) and the micro-batch snapshot rule of
    north_star.

Everything numeric runs in the library (tacg_coact_accumulate, tacg_affinity_swapgain, tacg_spectral_place,
gesr_build_replicas, tacg_eval_placement); this module only sorts a count vector and formats reports.

    python -m paper_2606_01007_b200.harness --config 2 [--tokens 65536] [--layers 4] [--gap] [--no-skew]   # JSON on stdout
"""
from __future__ import annotations

import argparse
import json
from typing import Dict, Optional, Tuple

import numpy as np
import torch

from . import binding as _b
from . import placement as _pl


def frequency_placement(D: torch.Tensor, ntok: torch.Tensor, capacity: int) -> np.ndarray:
    """The "Frequency" placement (PAPER.md:176 names it, nothing defines it; reading Q39 of DESIGN.md): per layer the
    experts are ranked by their pooled usage sum_f D[l,f,e]/max(1,N_f) (ties -> lower id) and partition m receives the
    ranks [m*capacity, (m+1)*capacity): frequently used experts share a partition.  int8[L,E]."""
    d = D.cpu().numpy().view(np.uint32).astype(np.float64)
    n = np.maximum(ntok.cpu().numpy().astype(np.float64), 1.0)
    pooled = (d / n[None, :, None]).sum(axis=1)                      # [L,E]
    L, E = pooled.shape
    out = np.empty((L, E), dtype=np.int8)
    for l in range(L):
        order = sorted(range(E), key=lambda e: (-pooled[l, e], e))
        for rank, e in enumerate(order):
            out[l, e] = rank // capacity
    return out


def build_placements(ctx: "_b.Context", cfg, D, Cm, ntok) -> Dict[str, Tuple[torch.Tensor, Optional[torch.Tensor]]]:
    """name -> (primary int8[L,E] tensor, replicas int8[L,E,r] tensor or None), all from the calibration counts."""
    dev = D.device
    L, F, E = D.shape
    P, cap = cfg.P, cfg.capacity
    out = {"baseline": (torch.from_numpy(_pl.default_placement(L, E, cap)).to(dev), None),
           "frequency": (torch.from_numpy(frequency_placement(D, ntok, cap)).to(dev), None)}
    for name, alpha in (("coactivation", 0.0), ("tacg", 0.25)):
        W = _b.tacg_affinity_swapgain(ctx, D, Cm, ntok, P, cap, None, alpha=alpha, want=("W",))["W"]
        out[name] = (_b.tacg_spectral_place(ctx, W, P, cap)["primary"], None)
    if cfg.r > 0 and cfg.n_rep > 0:
        primary = out["tacg"][0]
        replicas, _ = _b.gesr_build_replicas(ctx, D, Cm, ntok, P, cap, primary, cfg.n_rep, cfg.r)
        out["tacg+gesr"] = (primary, replicas)
    return out


def evaluate(ctx: "_b.Context", cfg, idx, fam, primary, replicas, microbatch=None) -> dict:
    """One placement over one trace: Comm (dispatch span per token, summed over layers), loads, Jain, MaxVio."""
    ev = _b.tacg_eval_placement(ctx, idx, fam, cfg.E, cfg.F, cfg.P, primary, replicas, theta=0.15, rho=0.995,
                                microbatch=cfg.microbatch if microbatch is None else microbatch)
    n = int(ev["ntok"].sum().item())
    span = int(ev["comm_span"].sum().item())
    fair = ev["fairness"][-1].cpu().numpy()
    return {"tokens": n, "comm_span_total": span, "comm": span / max(1, n), "jain": float(fair[0]),
            "maxvio": float(fair[1]), "load": ev["load"].cpu().numpy().astype(np.int64).sum(axis=0).tolist()}


def skew_report(ctx: "_b.Context", cfg, params, placements, N: int, seed: int, device="cuda") -> dict:
    """Every placement, held fixed, over the 13 online workloads (only the family stream changes; the expert choices
    follow the family, so the indices are drawn again per stream).  Comm. Red. is against "baseline" (Eq. 16)."""
    import tracegen
    report = {}
    for wi, wname in enumerate(tracegen.skew_workloads(cfg.F)):
        fam = tracegen.gen_family_workload(N, wname, cfg.F, seed + wi, device=device)
        idx = tracegen.gen_indices(cfg, params, fam, seed + 100 + wi, eval_trace=True, device=device)
        rows = {name: evaluate(ctx, cfg, idx, fam, pr, rp) for name, (pr, rp) in placements.items()}
        base = rows["baseline"]["comm"]
        for name, row in rows.items():
            row["comm_red_pct"] = 100.0 * (base - row["comm"]) / base if base > 0 else 0.0
        report[wname] = rows
    return report


def per_token_gap(ctx: "_b.Context", cfg, idx, fam, primary, replicas) -> dict:
    """f4: what the micro-batch snapshot of north_star changes against the literal per-token decay of Eq. 15."""
    lit = evaluate(ctx, cfg, idx, fam, primary, replicas, microbatch=1)
    snap = evaluate(ctx, cfg, idx, fam, primary, replicas, microbatch=cfg.microbatch)
    return {"per_token": lit, "microbatch": snap, "B": cfg.microbatch,
            "delta_comm_pct": 100.0 * (snap["comm"] - lit["comm"]) / lit["comm"] if lit["comm"] else 0.0,
            "delta_jain": snap["jain"] - lit["jain"], "delta_maxvio": snap["maxvio"] - lit["maxvio"]}


def main():
    import tracegen
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--tokens", type=int, default=65536, help="tokens per layer of the calibration and online traces")
    ap.add_argument("--layers", type=int, default=4)
    ap.add_argument("--gap", action="store_true", help="also the per-token against micro-batch comparison (f4)")
    ap.add_argument("--no-skew", action="store_true", help="skip the 13-workload sweep")
    args = ap.parse_args()
    base = tracegen.get_config(args.config)
    cfg = tracegen.scaled(base, N=args.tokens, N_eval=args.tokens, L=min(base.L, args.layers))
    params = tracegen.make_params(cfg)
    with _b.Context(0) as ctx:
        bi, bf = tracegen.gen_trace(cfg, params, device="cuda")
        co = _b.tacg_coact_accumulate(ctx, bi, bf, cfg.E, cfg.F)
        placements = build_placements(ctx, cfg, co["D"], co["C"], co["ntok"])
        out = {"config": cfg.name, "tokens": args.tokens, "layers": cfg.L,
               "skew": {} if args.no_skew else skew_report(ctx, cfg, params, placements, args.tokens, cfg.seed + 11)}
        if args.gap and "tacg+gesr" in placements:
            ei, ef = tracegen.gen_trace(cfg, params, eval_trace=True, device="cuda")
            pr, rp = placements["tacg+gesr"]
            out["per_token_gap"] = per_token_gap(ctx, cfg, ei, ef, pr, rp)
    for rows in out["skew"].values():
        for row in rows.values():
            row.pop("load", None)
    print(json.dumps(out))


if __name__ == "__main__":
    main()

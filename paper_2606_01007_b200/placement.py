"""Host-side placement driver (harness) -- consumes the library's outputs.

These are the consumers of the hot path, not part of it: a capacity-preserving best-swap
local search driven by the GPU swap gains (the "only if the move improves" test of
PAPER.md:124 applied to every pair), the whole offline stage of the method chained on the device
(`tacg_gesr_placement`: counts -> graph -> spectral-then-repair -> replicas by gesr_build_replicas).  All
E x E arithmetic stays in tacg_affinity_swapgain; the host only takes argmaxes.
"""
from __future__ import annotations

from typing import Optional, Tuple

import numpy as np
import torch

from . import binding as _b


def default_placement(L: int, E: int, capacity: int) -> np.ndarray:
    """primary[l,e] = e // capacity (the paper's 'Baseline' placement)."""
    return np.tile((np.arange(E) // capacity).astype(np.int8), (L, 1))


def local_search(ctx: "_b.Context", D, Cm, ntok, P: int, capacity: int, alpha: float = 0.25, tau: float = 1.0,
                 eps: float = 1e-6, max_swaps: Optional[int] = None,
                 primary0: Optional[np.ndarray] = None) -> Tuple[np.ndarray, np.ndarray]:
    """Best-swap local search on every layer at once.  Each round calls
    tacg_affinity_swapgain for all layers, copies gain/aff/W back and applies, per layer, the
    swap with the largest gain if it exceeds 1e-7 * sum|terms| (ties -> smallest (i,j)).
    Returns (primary int8[L,E], swaps per layer)."""
    L, F, E = D.shape
    primary = default_placement(L, E, capacity) if primary0 is None else primary0.astype(np.int8).copy()
    if max_swaps is None:
        max_swaps = 4 * E
    swaps = np.zeros(L, dtype=np.int64)
    active = np.ones(L, dtype=bool)
    dev = D.device
    ar = np.arange(E)
    for _ in range(max_swaps):
        out = _b.tacg_affinity_swapgain(ctx, D, Cm, ntok, P, capacity, torch.from_numpy(primary).to(dev),
                                        alpha=alpha, tau=tau, eps=eps, want=("W", "aff", "gain"))
        G = out["gain"].cpu().numpy()
        aff = out["aff"].cpu().numpy()
        W = out["W"].cpu().numpy()
        any_swap = False
        for l in np.nonzero(active)[0]:
            g = np.triu(G[l], 1)
            flat = int(np.argmax(g))            # first maximum = smallest (i,j)
            i, j = divmod(flat, E)
            best = float(g[i, j])
            a, b = int(primary[l, i]), int(primary[l, j])
            terms = abs(aff[l, i, b]) + abs(aff[l, j, a]) + abs(aff[l, i, a]) + abs(aff[l, j, b]) + 2 * abs(W[l, i, j])
            if a != b and best > 1e-7 * terms and best > 0:
                primary[l, i], primary[l, j] = b, a
                swaps[l] += 1
                any_swap = True
            else:
                active[l] = False
        if not any_swap:
            break
    return primary, swaps


def tacg_gesr_placement(ctx: "_b.Context", D, Cm, ntok, P: int, capacity: int, n_rep: int, r: int,
                        alpha: float = 0.25, tau: float = 1.0, eps: float = 1e-6, lambda1: float = 0.0,
                        lambda2: float = 0.0, refine: bool = False):
    """The offline stage of the method, every step on the device: the task-modulated
    graph W (Eq. 7-8), the spectral-then-repair primary placement (Eq. 9-10), optionally refined by the
    swap-gain local search, and the GESR replica table (Eq. 11-12).  Returns (primary int8[L,E] tensor,
    replicas int8[L,E,r] tensor or None)."""
    W = _b.tacg_affinity_swapgain(ctx, D, Cm, ntok, P, capacity, None, alpha=alpha, tau=tau, eps=eps, want=("W",))["W"]
    primary = _b.tacg_spectral_place(ctx, W, P, capacity)["primary"]
    if refine:
        refined, _ = local_search(ctx, D, Cm, ntok, P, capacity, alpha=alpha, tau=tau, eps=eps,
                                  primary0=primary.cpu().numpy())
        primary = torch.from_numpy(refined).to(D.device)
    replicas = None
    if r > 0 and n_rep > 0:
        replicas, _ = _b.gesr_build_replicas(ctx, D, Cm, ntok, P, capacity, primary, n_rep, r, lambda1=lambda1,
                                             lambda2=lambda2, alpha=alpha, tau=tau, eps=eps)
    return primary, replicas

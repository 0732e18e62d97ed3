"""Seeded trace sampling (torch, device-agnostic: CPU for tests, CUDA for full sizes).

The oracle and the library always consume THE SAME buffer produced here, so
parity never depends on regenerating a trace.  torch's CPU and CUDA generators
are different streams: a (config, seed) pair names one trace per device type.

Recipe:
  * small per-config parameters are drawn with numpy.random.default_rng(seed):
    expert popularity pi[l,f,:] (Dirichlet(a) or Zipf(s) over a random
    permutation), planted groups (a random partition of the experts of each
    layer into groups of `group_size`; config 1: one random perfect matching
    per family), family-specific group weights omega[l,f,:] ~ Dirichlet(0.5)
    (config 1: uniform), and `n_generic` generic expert ids per layer whose
    popularity is generic_mass/E for every family (rest rescaled);
  * family labels are i.i.d. from the mix;
  * per token of family f: with prob p_group pick a group g ~ omega[l,f] and
    take k of its members uniformly without replacement in random order (all of
    it when the group has exactly k members); otherwise take k experts without
    replacement from pi[l,f] (sequential draws, torch.multinomial).
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np
import torch

from .configs import TraceConfig


@dataclass
class TraceParams:
    pi: np.ndarray        # [L,F,E] float64, build-trace popularity
    pi_eval: np.ndarray   # [L,F,E] float64, eval-trace popularity (generic mass may differ)
    groups: np.ndarray    # [L,F,G,gs] int64 planted groups (same for all f except config 1)
    omega: np.ndarray     # [L,F,G] float64 group weights
    generic: np.ndarray   # [L,n_generic] int64


def _with_generic(pi: np.ndarray, generic: np.ndarray, mass_units: float, E: int) -> np.ndarray:
    """Set pi[l,f,g] = mass_units/E for generic ids g, rescale the rest to sum to 1."""
    out = pi.copy()
    L, F, _ = pi.shape
    ng = generic.shape[1]
    if ng == 0 or mass_units <= 0:
        return out
    gm = mass_units / E
    for l in range(L):
        g = generic[l]
        for f in range(F):
            rest = np.ones(E, dtype=bool)
            rest[g] = False
            s = out[l, f, rest].sum()
            out[l, f, rest] *= (1.0 - gm * ng) / s
            out[l, f, g] = gm
    return out


def make_params(cfg: TraceConfig, seed: Optional[int] = None) -> TraceParams:
    rng = np.random.default_rng(cfg.seed if seed is None else seed)
    L, F, E = cfg.L, cfg.F, cfg.E
    if cfg.popularity == "dirichlet":
        pi = rng.dirichlet(np.full(E, cfg.pop_param), size=(L, F))
        pi = np.maximum(pi, 1e-9)
        pi /= pi.sum(-1, keepdims=True)
    elif cfg.popularity == "zipf":
        base = np.arange(1, E + 1, dtype=np.float64) ** (-cfg.pop_param)
        base /= base.sum()
        pi = np.empty((L, F, E))
        for l in range(L):
            for f in range(F):
                pi[l, f, rng.permutation(E)] = base
    else:
        raise ValueError(cfg.popularity)
    gs = cfg.group_size
    G = E // gs
    groups = np.empty((L, F, G, gs), dtype=np.int64)
    for l in range(L):
        if cfg.name == "tiny":
            for f in range(F):                      # one perfect matching per family
                groups[l, f] = rng.permutation(E)[: G * gs].reshape(G, gs)
        else:
            part = rng.permutation(E)[: G * gs].reshape(G, gs)
            groups[l, :] = part[None]
    if cfg.name == "tiny":
        omega = np.full((L, F, G), 1.0 / G)
    else:
        omega = rng.dirichlet(np.full(G, 0.5), size=(L, F))
        omega = np.maximum(omega, 1e-9)
        omega /= omega.sum(-1, keepdims=True)
    generic = np.empty((L, cfg.n_generic), dtype=np.int64)
    for l in range(L):
        generic[l] = rng.choice(E, size=cfg.n_generic, replace=False)
    pi_b = _with_generic(pi, generic, cfg.generic_mass, E)
    pi_e = _with_generic(pi, generic, cfg.generic_mass_eval, E)
    return TraceParams(pi=pi_b, pi_eval=pi_e, groups=groups, omega=omega, generic=generic)


def _gen(device, seed: int) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed) & 0x7FFFFFFFFFFFFFFF)
    return g


def gen_family(N: int, mix, seed: int, device="cpu") -> torch.Tensor:
    """int8[N] family labels, i.i.d. from `mix`."""
    g = _gen(device, seed * 1_000_003 + 999_983)
    p = torch.tensor(mix, dtype=torch.float32, device=device)
    out = torch.empty(N, dtype=torch.int8, device=device)
    step = 1 << 22
    for s in range(0, N, step):
        n = min(step, N - s)
        out[s:s + n] = torch.multinomial(p, n, replacement=True, generator=g).to(torch.int8)
    return out


SKEW_SHARES = (0.6, 0.8)
BURST_SHARE = 0.15
BURST_FAMILIES = (2, 3)     # "math", "complex_reasoning" in the paper's family order


def skew_workloads(F: int = 4):
    """Names of the 13 online workloads of the paper's skew sweep: one
    balanced reference, F families x two single-family shares, two phase-shift streams, two
    bursty streams.  Only the family-label stream changes between them."""
    names = ["balanced"]
    names += [f"single:{f}:{s}" for f in range(F) for s in SKEW_SHARES]
    names += ["phase:up", "phase:down"]
    names += [f"burst:{f}" for f in BURST_FAMILIES if f < F]
    return names


def gen_family_workload(N: int, workload: str, F: int, seed: int, device="cpu",
                        phases: int = 8) -> torch.Tensor:
    """int8[N] family labels of one skew workload (the paper gives the suite in one sentence,
    PAPER.md:383; the numbers it leaves open are fixed here and listed in DESIGN.md Q32):
      balanced       i.i.d. uniform over the F families;
      single:f:s     i.i.d., family f with share s, the others (1-s)/(F-1) each;
      phase:up|down  the stream is cut into `phases` equal spans; span j is i.i.d. with family
                     j mod F (up) or F-1 - j mod F (down) at share 0.8;
      burst:f        the balanced stream with one contiguous span of 15 % of the tokens, starting
                     at 40 % of the stream, relabelled f.
    """
    kind, *rest = workload.split(":")
    if kind == "balanced":
        return gen_family(N, (1.0 / F,) * F, seed, device=device)
    if kind == "single":
        f, s = int(rest[0]), float(rest[1])
        mix = [(1.0 - s) / (F - 1)] * F
        mix[f] = s
        return gen_family(N, mix, seed, device=device)
    if kind == "phase":
        out = torch.empty(N, dtype=torch.int8, device=device)
        for j in range(phases):
            lo, hi = j * N // phases, (j + 1) * N // phases
            f = j % F if rest[0] == "up" else F - 1 - j % F
            mix = [0.2 / (F - 1)] * F
            mix[f] = 0.8
            out[lo:hi] = gen_family(hi - lo, mix, seed * 31 + j, device=device)
        return out
    if kind == "burst":
        out = gen_family(N, (1.0 / F,) * F, seed, device=device)
        lo = int(0.4 * N)
        out[lo:lo + int(BURST_SHARE * N)] = int(rest[0])
        return out
    raise ValueError(workload)


def gen_indices(cfg: TraceConfig, params: TraceParams, family: torch.Tensor, seed: int,
                eval_trace: bool = False, device="cpu", chunk: int = 1 << 20,
                out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """int16[L,N,k] top-k expert ids, k distinct per token."""
    L, E, k = cfg.L, cfg.E, cfg.k
    N = family.numel()
    gs = cfg.group_size
    if out is None:
        out = torch.empty((L, N, k), dtype=torch.int16, device=device)
    pi_np = params.pi_eval if eval_trace else params.pi
    for l in range(L):
        g = _gen(device, seed * 1_000_003 + l)
        pi = torch.tensor(pi_np[l], dtype=torch.float32, device=device)          # [F,E]
        omega = torch.tensor(params.omega[l], dtype=torch.float32, device=device)  # [F,G]
        groups = torch.tensor(params.groups[l], dtype=torch.int64, device=device)  # [F,G,gs]
        for s in range(0, N, chunk):
            n = min(chunk, N - s)
            fam = family[s:s + n].long()
            grp = torch.multinomial(omega[fam], 1, generator=g).squeeze(1)         # [n]
            members = groups[fam, grp]                                             # [n,gs]
            order = torch.rand((n, gs), generator=g, device=device).argsort(dim=1)[:, :k]
            from_group = members.gather(1, order)                                  # [n,k]
            from_pop = torch.multinomial(pi[fam], k, replacement=False, generator=g)
            use_group = torch.rand(n, generator=g, device=device) < cfg.p_group
            if gs < k:
                use_group = torch.zeros_like(use_group)
                from_group = from_pop
            idx = torch.where(use_group[:, None], from_group, from_pop)
            out[l, s:s + n] = idx.to(torch.int16)
    return out


def gen_trace(cfg: TraceConfig, params: Optional[TraceParams] = None, eval_trace: bool = False,
              device="cpu", seed: Optional[int] = None):
    """(indices int16[L,N,k], family int8[N]) for the build or the held-out eval trace."""
    if params is None:
        params = make_params(cfg)
    base = cfg.seed if seed is None else seed
    if eval_trace:
        base = base + 1
    N = cfg.N_eval if eval_trace else cfg.N
    mix = cfg.mix_eval if eval_trace else cfg.mix
    family = gen_family(N, mix, base, device=device)
    indices = gen_indices(cfg, params, family, base, eval_trace=eval_trace, device=device)
    return indices, family


def random_placement(E: int, P: int, capacity: int, L: int, seed: int) -> np.ndarray:
    """int8[L,E]: a uniformly random capacity-feasible primary map per layer (test input)."""
    assert E <= P * capacity
    rng = np.random.default_rng(seed)
    out = np.empty((L, E), dtype=np.int8)
    slots = np.repeat(np.arange(P, dtype=np.int8), capacity)
    for l in range(L):
        out[l] = rng.permutation(slots)[:E]
    return out


def random_replicas(primary: np.ndarray, P: int, r: int, n_rep: int, seed: int) -> np.ndarray:
    """int8[L,E,r]: for n_rep random experts per layer, r distinct non-primary partitions; -1 elsewhere."""
    rng = np.random.default_rng(seed)
    L, E = primary.shape
    out = np.full((L, E, max(r, 0)), -1, dtype=np.int8)
    if r == 0:
        return out
    for l in range(L):
        for e in rng.choice(E, size=min(n_rep, E), replace=False):
            others = [m for m in range(P) if m != primary[l, e]]
            nsec = min(r, len(others))
            if nsec > 0:
                nsec = int(rng.integers(1, nsec + 1))   # partially filled rows also occur
                out[l, e, :nsec] = rng.choice(others, size=nsec, replace=False)
    return out


def checksum64(t: torch.Tensor) -> int:
    """Order-sensitive 64-bit checksum of a tensor's bytes (wrapping int64 arithmetic)."""
    b = t.contiguous().view(torch.uint8).reshape(-1)
    pad = (-b.numel()) % 8
    if pad:
        b = torch.cat([b, torch.zeros(pad, dtype=torch.uint8, device=b.device)])
    w = b.view(torch.int64)
    total = 0
    step = 1 << 24
    for s in range(0, w.numel(), step):
        x = w[s:s + step]
        pos = torch.arange(s, s + x.numel(), dtype=torch.int64, device=x.device) * 2 + 1
        total = (total + int((x * pos).sum().item())) & 0xFFFFFFFFFFFFFFFF
    return total

"""The five workloads of BASELINE.json:configs, as data.

Config numbers follow BASELINE.json order (1 = Tiny ... 5 = distribution shift).
Fields marked (+) fill gaps BASELINE.json leaves open; they follow SURVEY.md
section 8(d) and are restated in DESIGN.md "Input recipe".
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Optional, Tuple


@dataclass(frozen=True)
class TraceConfig:
    name: str
    E: int                 # routed experts per layer
    k: int                 # top-k
    L: int                 # MoE layers
    F: int                 # task families (K in the paper)
    N: int                 # tokens per layer, build (calibration) trace
    N_eval: int            # tokens per layer, held-out eval trace
    P: int                 # partitions (simulated devices, M in the paper)
    capacity: int          # experts per partition (upper bound)
    mix: Tuple[float, ...]         # family mix of the build trace
    mix_eval: Tuple[float, ...]    # family mix of the eval trace
    popularity: str        # "dirichlet" or "zipf"
    pop_param: float       # Dirichlet concentration or Zipf exponent
    group_size: int        # planted group size
    p_group: float         # prob. a token draws its experts from a planted group
    n_generic: int         # generic experts per layer planted as shared across families
    generic_mass: float    # popularity of each generic expert, in units of 1/E (build)
    generic_mass_eval: float   # same, eval trace (config 5: x3)
    r: int                 # GESR secondary replicas per generic expert (0 = no GESR)
    n_rep: int             # generic experts replicated per layer
    microbatch: int        # GESR load-snapshot micro-batch B
    seed: int


CONFIGS = {
    1: TraceConfig(
        name="tiny", E=8, k=2, L=1, F=2, N=4096, N_eval=4096, P=4, capacity=2,
        mix=(0.5, 0.5), mix_eval=(0.5, 0.5), popularity="dirichlet", pop_param=0.5,
        group_size=2, p_group=0.7, n_generic=0, generic_mass=0.0, generic_mass_eval=0.0,
        r=0, n_rep=0, microbatch=256, seed=0),
    2: TraceConfig(
        name="moonlight_E64_k6_L26", E=64, k=6, L=26, F=4, N=262144, N_eval=262144,
        P=8, capacity=8, mix=(0.25,) * 4, mix_eval=(0.25,) * 4,
        popularity="dirichlet", pop_param=0.3, group_size=8, p_group=0.6,
        n_generic=0, generic_mass=0.0, generic_mass_eval=0.0,
        r=0, n_rep=0, microbatch=65536, seed=2000),
    3: TraceConfig(
        name="E128_k8_L48_gesr", E=128, k=8, L=48, F=4, N=1048576, N_eval=1048576,
        P=16, capacity=8, mix=(0.25,) * 4, mix_eval=(0.25,) * 4,
        popularity="dirichlet", pop_param=0.3, group_size=8, p_group=0.6,
        n_generic=4, generic_mass=4.0, generic_mass_eval=4.0,
        r=2, n_rep=4, microbatch=65536, seed=3000),
    4: TraceConfig(
        name="E256_k8_L58_zipf_gesr", E=256, k=8, L=58, F=4, N=4194304, N_eval=4194304,
        P=32, capacity=8, mix=(0.25,) * 4, mix_eval=(0.25,) * 4,
        popularity="zipf", pop_param=1.1, group_size=8, p_group=0.6,
        n_generic=8, generic_mass=4.0, generic_mass_eval=4.0,
        r=2, n_rep=8, microbatch=65536, seed=4000),
    5: TraceConfig(
        name="shift_E160_k6_L1", E=160, k=6, L=1, F=4, N=1048576, N_eval=16777216,
        P=16, capacity=10, mix=(0.4, 0.3, 0.2, 0.1), mix_eval=(0.1, 0.2, 0.3, 0.4),
        popularity="dirichlet", pop_param=0.3, group_size=8, p_group=0.6,
        n_generic=5, generic_mass=4.0, generic_mass_eval=12.0,
        r=3, n_rep=5, microbatch=65536, seed=5000),
}


def get_config(i: int) -> TraceConfig:
    return CONFIGS[int(i)]


def scaled(cfg: TraceConfig, N: Optional[int] = None, N_eval: Optional[int] = None,
           L: Optional[int] = None, microbatch: Optional[int] = None) -> TraceConfig:
    """Same shape, fewer tokens/layers (for parity cases the oracle finishes in seconds)."""
    kw = {}
    if N is not None:
        kw["N"] = int(N)
    if N_eval is not None:
        kw["N_eval"] = int(N_eval)
    if L is not None:
        kw["L"] = int(L)
    if microbatch is not None:
        kw["microbatch"] = int(microbatch)
    return replace(cfg, **kw)

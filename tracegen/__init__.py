"""Seeded synthetic routing-trace generator (inputs only).

This module serves BOTH the oracle (``oracle/``) and the CUDA path
(``paper_2606_01007_b200/``).  It holds none of the method's arithmetic: it
only draws top-k expert-index traces, family labels and random feasible
placements.  Neither ``oracle`` nor ``paper_2606_01007_b200`` is imported here.

What the traces stand in for: the paper measures on routing traces of
DeepSeek-MoE-16B, Qwen1.5-MoE-A2.7B and Moonlight-16B-A3B over nine public
datasets.  None of those models, datasets or traces is in
this container; the generator takes only their *shapes* (E, k, MoE layer
count, four task families, interleaved multi-task traffic; PAPER.md:23,
393-405 Table 5).  The recipe is stated in DESIGN.md "Input recipe".
"""
from .configs import TraceConfig, CONFIGS, get_config, scaled
from .generator import (
    TraceParams,
    make_params,
    gen_family,
    gen_family_workload,
    skew_workloads,
    gen_indices,
    gen_trace,
    random_placement,
    random_replicas,
    checksum64,
)

__all__ = [
    "TraceConfig", "CONFIGS", "get_config", "scaled", "TraceParams", "make_params",
    "gen_family", "gen_family_workload", "skew_workloads", "gen_indices", "gen_trace", "random_placement",
    "random_replicas", "checksum64",
]

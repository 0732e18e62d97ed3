"""paper_2606_01007_b200 -- B200-native hot path of TACG/GESR expert placement.

A thin ctypes binding (argument marshalling only) over libtacg.so, the C-ABI library of
hand-written sm_100a CUDA kernels declared in include/tacg.h.  torch is used for device
memory and streams only.  There is no CPU fallback: importing works without a GPU (so the
ABI can be inspected), but creating a Context without an sm_100 device raises.
"""
from .binding import (  # noqa: F401
    Context, TacgError, lib, lib_path, version,
    tacg_coact_accumulate, tacg_affinity_swapgain, gesr_select, tacg_eval_placement, gesr_build_replicas,
    tacg_spectral_place, tacg_family_divergence, tacg_eval_primary_noalloc, NOALLOC_SCRATCH_BYTES,
    TACG_ZERO_FIRST, TACG_VALIDATE, TACG_PATH_AUTO, TACG_PATH_HIST, TACG_PATH_MMA,
    TACG_PROF_COACT, TACG_PROF_AFFINITY, TACG_PROF_EVAL, TACG_PEAK_ATOMS_SPREAD, TACG_PEAK_ATOMS_RANDOM,
    TACG_PEAK_I8_TENSOR, EXPORTS,
)

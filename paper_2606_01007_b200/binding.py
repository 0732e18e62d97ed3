"""ctypes binding of libtacg.so: same names as include/tacg.h, marshalling only.

Every function takes torch CUDA tensors (or None) and passes their data_ptr() through;
shapes and dtypes are checked here, every step of the path runs in the library's kernels.
The convenience wrappers allocate the output tensors (device memory is torch's job) and
return them in a dict.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtacg.so")

TACG_ZERO_FIRST = 0x1
TACG_VALIDATE = 0x2
TACG_PATH_AUTO = 0x00
TACG_PATH_HIST = 0x10
TACG_PATH_MMA = 0x20
TACG_PROF_COACT, TACG_PROF_AFFINITY, TACG_PROF_EVAL = 0, 1, 2
TACG_PEAK_ATOMS_SPREAD, TACG_PEAK_ATOMS_RANDOM, TACG_PEAK_I8_TENSOR = 0, 1, 2

EXPORTS = (
    "tacg_create", "tacg_destroy", "tacg_strerror", "tacg_last_detail", "tacg_last_path",
    "tacg_launch_count", "tacg_version", "tacg_profile_enable", "tacg_profile_read", "tacg_measure_peak",
    "tacg_coact_accumulate", "tacg_affinity_swapgain",
    "gesr_select", "tacg_eval_placement", "gesr_build_replicas", "tacg_spectral_place", "tacg_family_divergence",
    "tacg_eval_primary_noalloc", "tacg_eval_primary_noalloc_prepare",
)

_lib = None


class TacgError(RuntimeError):
    def __init__(self, code: int, where: str, detail: str = ""):
        self.code = code
        msg = f"{where}: {lib().tacg_strerror(code).decode()} ({code})"
        if detail:
            msg += f" -- {detail}"
        super().__init__(msg)


def lib_path() -> str:
    return _SO


def lib():
    """Loads libtacg.so (built by paper_2606_01007_b200.build / __graft_entry__.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise FileNotFoundError(
                f"{_SO} is missing: run `python -m paper_2606_01007_b200.build` (there is no CPU fallback)")
        L = C.CDLL(_SO)
        vp, i32, i64, u32, f32, f64 = C.c_void_p, C.c_int, C.c_int64, C.c_uint32, C.c_float, C.c_double
        L.tacg_create.argtypes = [C.POINTER(vp), i32, vp]
        L.tacg_destroy.argtypes = [vp]
        L.tacg_strerror.argtypes = [i32]
        L.tacg_strerror.restype = C.c_char_p
        L.tacg_last_detail.argtypes = [vp, C.c_char_p, C.c_size_t]
        L.tacg_last_path.argtypes = [vp]
        L.tacg_launch_count.argtypes = [vp]
        L.tacg_launch_count.restype = i64
        L.tacg_version.restype = C.c_char_p
        L.tacg_profile_enable.argtypes = [vp, i32]
        L.tacg_profile_read.argtypes = [vp, i32, C.POINTER(f64), C.POINTER(i64)]
        L.tacg_measure_peak.argtypes = [vp, i32, C.POINTER(f64), C.POINTER(f64)]
        L.tacg_coact_accumulate.argtypes = [vp, vp, vp, i64, i32, i32, i32, i32, vp, vp, vp, u32]
        L.tacg_affinity_swapgain.argtypes = [vp, vp, vp, vp, i32, i32, i32, i32, i32, vp, f32, f32, f32,
                                             vp, vp, vp, vp]
        L.gesr_select.argtypes = [vp, vp, i64, i32, i32, i32, i32, vp, vp, i32, vp, f32, i64, vp, u32]
        L.gesr_build_replicas.argtypes = [vp, vp, vp, vp, i32, i32, i32, i32, i32, vp, f32, f32, f32, f32, f32,
                                          i32, i32, vp, vp]
        L.tacg_family_divergence.argtypes = [vp, vp, vp, vp, i32, i32, i32, i32, vp, vp]
        L.tacg_spectral_place.argtypes = [vp, vp, i32, i32, i32, i32, f64, i32, vp, vp, vp, vp]
        L.tacg_eval_placement.argtypes = [vp, vp, vp, i64, i32, i32, i32, i32, i32, vp, vp, i32, f32, f64,
                                          i64, i64, vp, vp, vp, vp, vp, vp, vp, vp, u32]
        L.tacg_eval_primary_noalloc_prepare.argtypes = [vp]
        L.tacg_eval_primary_noalloc.argtypes = [vp, vp, vp, i64, i32, i32, i32, i32, i32, vp, f64, i64,
                                                vp, vp, vp, vp, vp, vp, vp, vp]
        for name in EXPORTS:
            getattr(L, name)
        _lib = L
    return _lib


def version() -> str:
    return lib().tacg_version().decode()


def _ptr(t: Optional[torch.Tensor], dtype=None, name="tensor", numel: Optional[int] = None):
    """Device pointer of a tensor after checking where it lives, its layout, its dtype and (numel given) that it
    holds at least the elements the C call will touch -- a short tensor would be an out-of-bounds device access."""
    if t is None:
        return None
    if numel is not None and t.numel() < int(numel):
        raise ValueError(f"{name} has {t.numel()} elements, the call needs {int(numel)}")
    if not t.is_cuda:
        raise ValueError(f"{name} must be a CUDA tensor (the library has no CPU path)")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"{name} must be {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _within_limits(k=1, L=1, E=1, F=1, P=1, r=0, N=0) -> bool:
    """The ABI limits of include/tacg.h.  Outside them the library itself refuses the call (TACG_ERR_SHAPE) before
    touching any buffer, so the binding leaves the error to it and checks buffer sizes only inside them."""
    return 1 <= k <= 16 and L >= 1 and 1 <= E <= 512 and 1 <= F <= 8 and 1 <= P <= 64 and 0 <= r <= 8 and N >= 0


class Context:
    """tacg_ctx bound to a device and a torch stream (default: the current stream)."""

    def __init__(self, device: int = 0, stream: Optional[torch.cuda.Stream] = None):
        self._h = C.c_void_p()
        self.device = int(device)
        if stream is None and torch.cuda.is_available():
            stream = torch.cuda.current_stream(self.device)
        self.stream = stream
        sp = C.c_void_p(stream.cuda_stream) if stream is not None else None
        rc = lib().tacg_create(C.byref(self._h), self.device, sp)
        if rc != 0:
            self._h = C.c_void_p()
            raise TacgError(rc, "tacg_create")

    def close(self):
        if self._h:
            lib().tacg_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def detail(self) -> str:
        buf = C.create_string_buffer(256)
        lib().tacg_last_detail(self._h, buf, 256)
        return buf.value.decode(errors="replace")

    def last_path(self) -> int:
        return int(lib().tacg_last_path(self._h))

    def launch_count(self) -> int:
        return int(lib().tacg_launch_count(self._h))

    def profile_enable(self, on: bool = True):
        self.check(lib().tacg_profile_enable(self._h, 1 if on else 0), "tacg_profile_enable")

    def profile_read(self, slot: int):
        """(total_ms, launches) of the slot's kernels since the last read (synchronises their events)."""
        ms, n = C.c_double(0.0), C.c_int64(0)
        self.check(lib().tacg_profile_read(self._h, int(slot), C.byref(ms), C.byref(n)), "tacg_profile_read")
        return ms.value, n.value

    def measure_peak(self, which: int):
        """(units per second, units per clock and SM) of one of the TACG_PEAK_* micro-benchmarks."""
        a, b = C.c_double(0.0), C.c_double(0.0)
        self.check(lib().tacg_measure_peak(self._h, int(which), C.byref(a), C.byref(b)), "tacg_measure_peak")
        return a.value, b.value

    def check(self, rc: int, where: str):
        if rc != 0:
            raise TacgError(rc, where, self.detail())

    def _enter(self):
        """The library enqueues on the stream the context was created with; torch allocates (and frees) the caller's
        tensors on the CURRENT stream.  Using the context under another stream would race silently, so refuse."""
        if self.stream is not None and torch.cuda.current_stream(self.device) != self.stream:
            raise ValueError("this tacg Context is bound to another CUDA stream than the current one: create one "
                             "Context per stream (tacg.Context(device, stream))")

    # ---- raw calls: same names and argument order as include/tacg.h ----
    def tacg_coact_accumulate(self, indices, family, N, k, L, E, F, D, Cm, ntok, flags=0) -> int:
        self._enter()
        ok = _within_limits(k=k, L=L, E=E, F=F, N=N)
        n = lambda v: v if ok else None
        return lib().tacg_coact_accumulate(
            self._h, _ptr(indices, torch.int16, "indices", n(L * N * k)), _ptr(family, torch.int8, "family", n(N)),
            int(N), int(k), int(L), int(E), int(F), _ptr(D, torch.int32, "D", n(L * F * E)),
            _ptr(Cm, torch.int32, "C", n(L * F * E * E)), _ptr(ntok, torch.int64, "ntok", n(F)), int(flags))

    def tacg_affinity_swapgain(self, D, Cm, ntok, L, E, F, P, capacity, primary, alpha, tau, eps,
                               pref, W, aff, gain) -> int:
        self._enter()
        ok = _within_limits(L=L, E=E, F=F, P=max(P, 1))
        n = lambda v: v if ok else None
        return lib().tacg_affinity_swapgain(
            self._h, _ptr(D, torch.int32, "D", n(L * F * E)), _ptr(Cm, torch.int32, "C", n(L * F * E * E)),
            _ptr(ntok, torch.int64, "ntok", n(F)), int(L), int(E), int(F), int(P), int(capacity),
            _ptr(primary, torch.int8, "primary", n(L * E)), float(alpha), float(tau), float(eps),
            _ptr(pref, torch.float32, "pref", n(L * E * F)), _ptr(W, torch.float32, "W", n(L * E * E)),
            _ptr(aff, torch.float32, "aff", n(L * E * P)), _ptr(gain, torch.float32, "gain", n(L * E * E)))

    def gesr_build_replicas(self, D, Cm, ntok, L, E, F, P, capacity, primary, alpha, tau, eps, lambda1, lambda2,
                            n_rep, r, replicas, terms) -> int:
        self._enter()
        ok = _within_limits(L=L, E=E, F=F, P=P, r=r)
        n = lambda v: v if ok else None
        return lib().gesr_build_replicas(
            self._h, _ptr(D, torch.int32, "D", n(L * F * E)), _ptr(Cm, torch.int32, "C", n(L * F * E * E)),
            _ptr(ntok, torch.int64, "ntok", n(F)), int(L), int(E), int(F), int(P), int(capacity),
            _ptr(primary, torch.int8, "primary", n(L * E)), float(alpha), float(tau), float(eps), float(lambda1),
            float(lambda2), int(n_rep), int(r), _ptr(replicas, torch.int8, "replicas", n(L * E * max(r, 0))),
            _ptr(terms, torch.float32, "terms", n(L * E * 4)))

    def tacg_family_divergence(self, D, Cm, ntok, L, E, F, topk, frob, jaccard) -> int:
        self._enter()
        ok = _within_limits(L=L, E=E, F=F)
        n = lambda v: v if ok else None
        return lib().tacg_family_divergence(
            self._h, _ptr(D, torch.int32, "D", n(L * F * E)), _ptr(Cm, torch.int32, "C", n(L * F * E * E)),
            _ptr(ntok, torch.int64, "ntok", n(F)), int(L), int(E), int(F), int(topk),
            _ptr(frob, torch.float32, "frob", n((L + 1) * F * F)), _ptr(jaccard, torch.float32, "jaccard", n((L + 1) * F * F)))

    def tacg_spectral_place(self, W, L, E, P, capacity, jitter, kmeans_iters, labels_in, primary, labels0, embed) -> int:
        self._enter()
        ok = _within_limits(L=L, E=E, P=P)
        n = lambda v: v if ok else None
        return lib().tacg_spectral_place(
            self._h, _ptr(W, torch.float32, "W", n(L * E * E)), int(L), int(E), int(P), int(capacity), float(jitter),
            int(kmeans_iters), _ptr(labels_in, torch.int8, "labels_in", n(L * E)), _ptr(primary, torch.int8, "primary", n(L * E)),
            _ptr(labels0, torch.int8, "labels0", n(L * E)), _ptr(embed, torch.float64, "embed", n(L * E * P)))

    def gesr_select(self, indices, N, k, L, E, P, primary, replicas, r, load_snapshot, theta,
                    token_offset, serve, flags=0) -> int:
        self._enter()
        ok = _within_limits(k=k, L=L, E=E, P=P, r=r, N=N)
        n = lambda v: v if ok else None
        return lib().gesr_select(
            self._h, _ptr(indices, torch.int16, "indices", n(L * N * k)), int(N), int(k), int(L), int(E), int(P),
            _ptr(primary, torch.int8, "primary", n(L * E)), _ptr(replicas, torch.int8, "replicas", n(L * E * max(r, 0))), int(r),
            _ptr(load_snapshot, torch.float64, "load_snapshot", n(L * P)), float(theta), int(token_offset),
            _ptr(serve, torch.int8, "serve", n(L * N * k)), int(flags))

    def tacg_eval_placement(self, indices, family, N, k, L, E, F, P, primary, replicas, r, theta, rho,
                            microbatch, token_offset, load_state, load, comm_span, comm_remote, ntok,
                            fairness, cost_per_token, serve, flags=0) -> int:
        self._enter()
        ok = _within_limits(k=k, L=L, E=E, F=F, P=P, r=r, N=N)
        n = lambda v: v if ok else None
        return lib().tacg_eval_placement(
            self._h, _ptr(indices, torch.int16, "indices", n(L * N * k)), _ptr(family, torch.int8, "family", n(N)),
            int(N), int(k), int(L), int(E), int(F), int(P), _ptr(primary, torch.int8, "primary", n(L * E)),
            _ptr(replicas, torch.int8, "replicas", n(L * E * max(r, 0))), int(r), float(theta), float(rho), int(microbatch),
            int(token_offset), _ptr(load_state, torch.float64, "load_state", n(L * P)),
            _ptr(load, torch.int64, "load", n(L * P)), _ptr(comm_span, torch.int64, "comm_span", n(L * F)),
            _ptr(comm_remote, torch.int64, "comm_remote", n(L * F)), _ptr(ntok, torch.int64, "ntok", n(F)),
            _ptr(fairness, torch.float32, "fairness", n((L + 1) * 3)), _ptr(cost_per_token, torch.uint8, "cost_per_token", n(L * N)),
            _ptr(serve, torch.int8, "serve", n(L * N * k)), int(flags))

    def tacg_eval_primary_noalloc_prepare(self) -> int:
        self._enter()
        return lib().tacg_eval_primary_noalloc_prepare(self._h)

    def tacg_eval_primary_noalloc(self, indices, family, N, k, L, E, F, P, primary, rho, token_offset, load_state,
                                  load, comm_span, comm_remote, ntok, fairness, cost_per_token, serve) -> int:
        self._enter()
        ok = _within_limits(k=k, L=L, E=E, F=F, P=P, r=0, N=N)
        n = lambda v: v if ok else None
        return lib().tacg_eval_primary_noalloc(
            self._h, _ptr(indices, torch.int16, "indices", n(L * N * k)), _ptr(family, torch.int8, "family", n(N)),
            int(N), int(k), int(L), int(E), int(F), int(P), _ptr(primary, torch.int8, "primary", n(L * E)),
            float(rho), int(token_offset), _ptr(load_state, torch.float64, "load_state", n(L * P)),
            _ptr(load, torch.int64, "load", n(L * P)), _ptr(comm_span, torch.int64, "comm_span", n(L * F)),
            _ptr(comm_remote, torch.int64, "comm_remote", n(L * F)), _ptr(ntok, torch.int64, "ntok", n(F)),
            _ptr(fairness, torch.float32, "fairness", n((L + 1) * 3)),
            _ptr(cost_per_token, torch.uint8, "cost_per_token", n(L * N)), _ptr(serve, torch.int8, "serve", n(L * N * k)))


# ---- convenience wrappers: allocate outputs with torch, call, return a dict ----
# uint32 / uint64 device buffers are held as torch int32 / int64 tensors (same bits).

def tacg_coact_accumulate(ctx: Context, indices, family, E: int, F: int, D=None, Cm=None, ntok=None,
                          flags: int = TACG_ZERO_FIRST):
    L, N, k = indices.shape
    dev = indices.device
    if D is None:
        D = torch.empty((L, F, E), dtype=torch.int32, device=dev)
        flags |= TACG_ZERO_FIRST
    if Cm is None:
        Cm = torch.empty((L, F, E, E), dtype=torch.int32, device=dev)
        flags |= TACG_ZERO_FIRST
    if ntok is None:
        ntok = torch.empty((F,), dtype=torch.int64, device=dev)
        flags |= TACG_ZERO_FIRST
    ctx.check(ctx.tacg_coact_accumulate(indices, family, N, k, L, E, F, D, Cm, ntok, flags),
              "tacg_coact_accumulate")
    return dict(D=D, C=Cm, ntok=ntok)


def tacg_affinity_swapgain(ctx: Context, D, Cm, ntok, P: int, capacity: int, primary, alpha=0.25, tau=1.0,
                           eps=1e-6, want=("pref", "W", "aff", "gain")):
    L, F, E = D.shape
    dev = D.device
    out = dict(pref=None, W=None, aff=None, gain=None)
    if "pref" in want:
        out["pref"] = torch.empty((L, E, F), dtype=torch.float32, device=dev)
    if "W" in want:
        out["W"] = torch.empty((L, E, E), dtype=torch.float32, device=dev)
    if "aff" in want and primary is not None:
        out["aff"] = torch.empty((L, E, P), dtype=torch.float32, device=dev)
    if "gain" in want and primary is not None:
        out["gain"] = torch.empty((L, E, E), dtype=torch.float32, device=dev)
    ctx.check(ctx.tacg_affinity_swapgain(D, Cm, ntok, L, E, F, P, capacity, primary, alpha, tau, eps,
                                         out["pref"], out["W"], out["aff"], out["gain"]),
              "tacg_affinity_swapgain")
    return out


def gesr_build_replicas(ctx: Context, D, Cm, ntok, P: int, capacity: int, primary, n_rep: int, r: int,
                        lambda1: float = 0.0, lambda2: float = 0.0, alpha=0.25, tau=1.0, eps=1e-6):
    """Eq. 11 scores and the Eq. 12 replica table on the device: returns (replicas int8[L,E,r],
    terms float32[L,E,4] = (score, Cent, Cons, Spec))."""
    L, F, E = D.shape
    replicas = torch.empty((L, E, r), dtype=torch.int8, device=D.device)
    terms = torch.empty((L, E, 4), dtype=torch.float32, device=D.device)
    ctx.check(ctx.gesr_build_replicas(D, Cm, ntok, L, E, F, P, capacity, primary, alpha, tau, eps, lambda1, lambda2,
                                      n_rep, r, replicas, terms), "gesr_build_replicas")
    return replicas, terms


def tacg_family_divergence(ctx: Context, D, Cm, ntok, topk: int = 64):
    """Activation Frobenius distance and top-k pair Jaccard overlap between task families:
    returns (frob float32[L+1,F,F], jaccard float32[L+1,F,F]); row L = whole model."""
    L, F, E = D.shape
    frob = torch.empty((L + 1, F, F), dtype=torch.float32, device=D.device)
    jac = torch.empty((L + 1, F, F), dtype=torch.float32, device=D.device)
    ctx.check(ctx.tacg_family_divergence(D, Cm, ntok, L, E, F, topk, frob, jac), "tacg_family_divergence")
    return frob, jac


def tacg_spectral_place(ctx: Context, W, P: int, capacity: int, jitter: float = 1e-6, kmeans_iters: int = 100,
                        labels_in=None, want_embed: bool = False):
    """Spectral-then-repair primary placement of every layer of W float32[L,E,E]:
    returns dict(primary int8[L,E], labels0 int8[L,E], embed float64[L,E,P] or None)."""
    L, E, _ = W.shape
    primary = torch.empty((L, E), dtype=torch.int8, device=W.device)
    labels0 = torch.empty((L, E), dtype=torch.int8, device=W.device)
    embed = torch.empty((L, E, P), dtype=torch.float64, device=W.device) if want_embed else None
    ctx.check(ctx.tacg_spectral_place(W, L, E, P, capacity, jitter, kmeans_iters, labels_in, primary, labels0, embed),
              "tacg_spectral_place")
    return dict(primary=primary, labels0=labels0, embed=embed)


def gesr_select(ctx: Context, indices, E: int, P: int, primary, replicas, load_snapshot, theta: float,
                token_offset: int = 0, flags: int = 0):
    L, N, k = indices.shape
    r = 0 if replicas is None else replicas.shape[2]
    serve = torch.empty((L, N, k), dtype=torch.int8, device=indices.device)
    ctx.check(ctx.gesr_select(indices, N, k, L, E, P, primary, replicas if r else None, r, load_snapshot,
                              theta, token_offset, serve, flags), "gesr_select")
    return serve


def tacg_eval_placement(ctx: Context, indices, family, E: int, F: int, P: int, primary, replicas=None,
                        theta: float = 0.15, rho: float = 0.995, microbatch: int = 0, token_offset: int = 0,
                        load_state=None, want_cost: bool = False, want_serve: bool = False, flags: int = 0):
    L, N, k = indices.shape
    dev = indices.device
    r = 0 if replicas is None else replicas.shape[2]
    out = dict(
        load=torch.empty((L, P), dtype=torch.int64, device=dev),
        comm_span=torch.empty((L, F), dtype=torch.int64, device=dev),
        comm_remote=torch.empty((L, F), dtype=torch.int64, device=dev),
        ntok=torch.empty((F,), dtype=torch.int64, device=dev),
        fairness=torch.empty((L + 1, 3), dtype=torch.float32, device=dev),
        cost=torch.empty((L, N), dtype=torch.uint8, device=dev) if want_cost else None,
        serve=torch.empty((L, N, k), dtype=torch.int8, device=dev) if want_serve else None,
        load_state=load_state,
    )
    ctx.check(ctx.tacg_eval_placement(indices, family, N, k, L, E, F, P, primary, replicas if r else None, r,
                                      theta, rho, microbatch, token_offset, load_state, out["load"],
                                      out["comm_span"], out["comm_remote"], out["ntok"], out["fairness"],
                                      out["cost"], out["serve"], flags), "tacg_eval_placement")
    return out


NOALLOC_SCRATCH_BYTES = 8 << 20      # TACG_NOALLOC_SCRATCH_BYTES of include/tacg.h


def tacg_eval_primary_noalloc(ctx: Context, indices, family, E: int, F: int, P: int, primary, out: dict,
                              rho: float = 0.995, token_offset: int = 0, load_state=None):
    """tacg_eval_placement without replicas through the entry point that allocates nothing: the caller passes every
    output in `out` (keys load, comm_span, comm_remote, ntok, fairness; optional cost, serve), this wrapper creates no
    tensor.  The library's scratch for it is a fixed device array of NOALLOC_SCRATCH_BYTES shared by all calls."""
    L, N, k = indices.shape
    ctx.check(ctx.tacg_eval_primary_noalloc(indices, family, N, k, L, E, F, P, primary, rho, token_offset, load_state,
                                            out["load"], out["comm_span"], out["comm_remote"], out["ntok"],
                                            out["fairness"], out.get("cost"), out.get("serve")),
              "tacg_eval_primary_noalloc")
    return out

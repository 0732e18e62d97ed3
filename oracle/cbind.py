"""ctypes binding of oracle/tacg_oracle.c -- TEST INFRASTRUCTURE ONLY.

`build()` compiles the C oracle with gcc (-O2 -ffp-contract=off -fopenmp) into
oracle/libtacg_oracle.so; the functions below marshal numpy arrays only.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tacg_oracle.c")
_SO = os.path.join(_HERE, "libtacg_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c11",
               "-o", _SO, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
        _lib.orc_threads.restype = C.c_int
    return _lib


def threads() -> int:
    return int(lib().orc_threads())


def set_threads(n: int) -> None:
    lib().orc_set_threads(C.c_int(n))


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _c(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def coact(indices, family, E: int, F: int, D=None, Cm=None, ntok=None):
    indices = _c(indices, np.int16)
    family = _c(family, np.int8)
    L, N, k = indices.shape
    if D is None:
        D = np.zeros((L, F, E), dtype=np.uint32)
    if Cm is None:
        Cm = np.zeros((L, F, E, E), dtype=np.uint32)
    if ntok is None:
        ntok = np.zeros(F, dtype=np.uint64)
    rc = lib().orc_coact(_p(indices), _p(family), C.c_int64(N), C.c_int(k), C.c_int(L), C.c_int(E),
                         C.c_int(F), _p(D), _p(Cm), _p(ntok))
    assert rc == 0
    return D, Cm, ntok


def affinity_swapgain(D, Cm, ntok, P: int, primary, alpha=0.25, tau=1.0, eps=1e-6):
    D = _c(D, np.uint32)
    Cm = _c(Cm, np.uint32)
    ntok = _c(ntok, np.uint64)
    L, F, E = D.shape
    primary = _c(primary, np.int8)
    pref = np.zeros((L, E, F))
    W = np.zeros((L, E, E))
    aff = np.zeros((L, E, P))
    gain = np.zeros((L, E, E))
    rc = lib().orc_affinity_swapgain(_p(D), _p(Cm), _p(ntok), C.c_int(L), C.c_int(E), C.c_int(F),
                                     C.c_int(P), _p(primary), C.c_double(alpha), C.c_double(tau),
                                     C.c_double(eps), _p(pref), _p(W), _p(aff), _p(gain))
    assert rc == 0
    return dict(pref=pref, W=W, aff=aff, gain=gain)


def gesr_select(indices, E: int, P: int, primary, replicas, load_snapshot, theta: float,
                token_offset: int = 0):
    indices = _c(indices, np.int16)
    L, N, k = indices.shape
    primary = _c(primary, np.int8)
    r = 0 if replicas is None else replicas.shape[2]
    replicas = None if replicas is None or r == 0 else _c(replicas, np.int8)
    snap = _c(load_snapshot, np.float64)
    serve = np.zeros((L, N, k), dtype=np.int8)
    rc = lib().orc_gesr_select(_p(indices), C.c_int64(N), C.c_int(k), C.c_int(L), C.c_int(E),
                               C.c_int(P), _p(primary), _p(replicas), C.c_int(r), _p(snap),
                               C.c_float(theta), C.c_int64(token_offset), _p(serve))
    assert rc == 0
    return serve


def eval_placement(indices, family, E: int, F: int, P: int, primary, replicas=None,
                   theta: float = 0.15, rho: float = 0.995, microbatch: int = 0,
                   load_state=None, token_offset: int = 0, want_cost: bool = False,
                   want_serve: bool = False):
    indices = _c(indices, np.int16)
    family = _c(family, np.int8)
    L, N, k = indices.shape
    primary = _c(primary, np.int8)
    r = 0 if replicas is None else replicas.shape[2]
    replicas = None if replicas is None or r == 0 else _c(replicas, np.int8)
    state = None if load_state is None else np.array(load_state, dtype=np.float64, order="C")
    load = np.zeros((L, P), dtype=np.uint64)
    span = np.zeros((L, F), dtype=np.uint64)
    remote = np.zeros((L, F), dtype=np.uint64)
    ntok = np.zeros(F, dtype=np.uint64)
    fair = np.zeros((L + 1, 3), dtype=np.float64)
    cost = np.zeros((L, N), dtype=np.uint8) if want_cost else None
    serve = np.zeros((L, N, k), dtype=np.int8) if want_serve else None
    rc = lib().orc_eval(_p(indices), _p(family), C.c_int64(N), C.c_int(k), C.c_int(L), C.c_int(E),
                        C.c_int(F), C.c_int(P), _p(primary), _p(replicas), C.c_int(r),
                        C.c_float(theta), C.c_double(rho), C.c_int64(microbatch),
                        C.c_int64(token_offset), _p(state), _p(load), _p(span), _p(remote),
                        _p(ntok), _p(fair), _p(cost), _p(serve))
    assert rc == 0
    return dict(load=load, comm_span=span, comm_remote=remote, ntok=ntok, fairness=fair,
                cost=cost, serve=serve, load_state=state)

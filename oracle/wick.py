"""ctypes loader for tier W (oracle/wick.c).  TEST INFRASTRUCTURE ONLY (see nbs_oracle.py)."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

from .nbs_oracle import BARYONS

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libnbs_wick.so")
_lib = None


def build(force: bool = False) -> str:
    src = os.path.join(_HERE, "wick.c")
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c11", "-o", _SO, src, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.wick_fourpt.restype = ctypes.c_int
    return _lib


def wick_fourpt(L: int, S: dict, ch, spins, rlist=None) -> np.ndarray:
    """Brute-force F[r, ispin] for channel ch = (B1,B2,B3,B4) and spin tuples (a1,a2,a3,a4)."""
    lib = _load()
    V = L ** 3
    rlist = np.arange(V, dtype=np.int32) if rlist is None else np.asarray(rlist, dtype=np.int32)
    nterm = np.zeros(4, dtype=np.int32)
    coef = np.zeros((4, 3), dtype=np.float64)
    flav = np.zeros((4, 3, 3), dtype=np.int32)
    for i, b in enumerate(ch):
        terms = BARYONS[b][1]
        nterm[i] = len(terms)
        for t, (k, f) in enumerate(terms):
            coef[i, t] = k
            flav[i, t] = ["uds".index(c) for c in f]
    spins = np.ascontiguousarray(np.asarray(spins, dtype=np.int32).reshape(-1, 4))
    out = np.zeros((len(rlist), len(spins)), dtype=np.complex128)
    arrs = [np.ascontiguousarray(S[f], dtype=np.complex128) for f in "uds"]
    p = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    rc = lib.wick_fourpt(ctypes.c_int(L), p(arrs[0]), p(arrs[1]), p(arrs[2]), p(nterm), p(coef), p(flav),
                         ctypes.c_int(len(spins)), p(spins), ctypes.c_int(len(rlist)), p(rlist), p(out))
    assert rc == 0
    return out

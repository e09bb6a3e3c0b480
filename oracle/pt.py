"""ORACLE — TEST INFRASTRUCTURE ONLY (see the header of pt_oracle.cpp).

ctypes loader for the plain C++ implementation of the paper's approximate counter (Algorithm 2,
PAPER.md:291-319).  Same import rules as the rest of ``oracle/``.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
import threading

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pt_oracle.cpp")
_SO = os.path.join(_HERE, "libpt_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    with _lock:
        if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
            tmp = _SO + ".tmp.%d" % os.getpid()
            subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", tmp, _SRC])
            os.replace(tmp, _SO)
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        u64, u64p, dp = ctypes.c_uint64, ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_double)
        lib.pt_run.argtypes = [ctypes.c_int, ctypes.c_int, dp, ctypes.c_int, u64, u64, u64, u64, u64p, u64p, u64p]
        lib.pt_run.restype = ctypes.c_int
        lib.pt_ratios.argtypes = [ctypes.c_int, ctypes.c_int, dp, ctypes.c_int, u64p, dp]
        lib.pt_ratios.restype = ctypes.c_double
        lib.pt_density_of_states.argtypes = [ctypes.c_int, ctypes.c_int, u64p]
        lib.pt_density_of_states.restype = ctypes.c_int
        lib.pt_draw.argtypes = [u64, u64]
        lib.pt_draw.restype = u64
        _lib = lib
    return _lib


def draw(seed: int, ctr: int) -> int:
    return int(_load().pt_draw(seed, ctr))


def run(kind: int, n: int, betas, replicas: int, iterations: int, seed: int, burn_in: int = 0):
    """Returns (hist[level][E], moves accepted per level, exchanges accepted per level) as lists of ints."""
    M, N = len(betas), 2 * n
    b = (ctypes.c_double * M)(*betas)
    hist = (ctypes.c_uint64 * (M * (N + 1)))()
    mv = (ctypes.c_uint64 * M)()
    sw = (ctypes.c_uint64 * M)()
    rc = _load().pt_run(kind, n, b, M, replicas, iterations, burn_in, seed, hist, mv, sw)
    assert rc == 0, rc
    return ([[int(hist[j * (N + 1) + e]) for e in range(N + 1)] for j in range(M)],
            [int(v) for v in mv], [int(v) for v in sw])


def ratios(kind: int, n: int, betas, hist):
    """(ratios per level, log of the estimated number of E = 0 configurations)."""
    M, N = len(betas), 2 * n
    b = (ctypes.c_double * M)(*betas)
    flat = (ctypes.c_uint64 * (M * (N + 1)))(*[v for row in hist for v in row])
    out = (ctypes.c_double * M)()
    logz = _load().pt_ratios(kind, n, b, M, flat, out)
    return [float(v) for v in out], float(logz)


def density_of_states(kind: int, n: int):
    g = (ctypes.c_uint64 * (2 * n + 1))()
    rc = _load().pt_density_of_states(kind, n, g)
    assert rc == 0, rc
    return [int(v) for v in g]


def exact_ratio(g, beta_lo: float, beta_hi: float) -> float:
    """Z(beta_hi)/Z(beta_lo) from a density of states (beta_hi may be math.inf)."""
    z = lambda b: sum(c * (math.exp(-b * e) if b != math.inf else (1.0 if e == 0 else 0.0)) for e, c in enumerate(g))
    return z(beta_hi) / z(beta_lo)

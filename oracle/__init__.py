"""ORACLE — TEST INFRASTRUCTURE ONLY (see the header of godfrey_oracle.cpp).

ctypes loader for the plain C++ oracle.  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package; the product
package ``paper_1507_00315_b200`` never does, and this package never imports it.

All results cross the boundary as decimal strings and are returned as Python ints.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "godfrey_oracle.cpp")
_SO = os.path.join(_HERE, "libgodfrey_oracle.so")
_lock = threading.Lock()
_lib = None

SKOLEM, LANGFORD = 0, 1
_CAP = 256


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (plain -O2, no tuning flags)."""
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
        u64, u32p = ctypes.c_uint64, ctypes.POINTER(ctypes.c_uint32)
        lib.godfrey_term.argtypes = [ctypes.c_int, ctypes.c_int, u64, ctypes.c_char_p, ctypes.c_size_t]
        lib.godfrey_term.restype = ctypes.c_int
        lib.godfrey_F.argtypes = lib.godfrey_term.argtypes
        lib.godfrey_F.restype = ctypes.c_int
        lib.godfrey_range.argtypes = [ctypes.c_int, ctypes.c_int, u64, u64, ctypes.c_char_p, ctypes.c_size_t,
                                      ctypes.POINTER(u64), u32p, ctypes.c_int, u32p]
        lib.godfrey_range.restype = ctypes.c_int
        lib.brute_count.argtypes = [ctypes.c_int, ctypes.c_int]
        lib.brute_count.restype = u64
        lib.brute_list.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_int), ctypes.c_int]
        lib.brute_list.restype = u64
        _lib = lib
    return _lib


def _xbits(x) -> int:
    """x = sequence of +1/-1 for positions 1..2n  ->  bit (p-1) set iff x_p = -1."""
    v = 0
    for p, xp in enumerate(x, start=1):
        assert xp in (1, -1)
        if xp == -1:
            v |= 1 << (p - 1)
    return v


def term(kind: int, n: int, x) -> int:
    """signX * F(n, X) for one sign vector (Algorithm 1's loop body)."""
    buf = ctypes.create_string_buffer(_CAP)
    rc = _load().godfrey_term(kind, n, _xbits(x), buf, _CAP)
    assert rc == 0, rc
    return int(buf.value)


def F(kind: int, n: int, x) -> int:
    """Godfrey's polynomial F(n, X) at one sign vector."""
    buf = ctypes.create_string_buffer(_CAP)
    rc = _load().godfrey_F(kind, n, _xbits(x), buf, _CAP)
    assert rc == 0, rc
    return int(buf.value)


def range_sum(kind: int, n: int, index_begin: int, index_end: int, moduli=()):
    """Sum of terms over indices [index_begin, index_end) of the 2^{2n} sign vectors.

    Returns (exact signed sum, number of non-zero terms, residues mod each modulus).
    Index convention: bit b of the index <-> position 2n-b, bit set <-> x = -1.
    """
    lib = _load()
    buf = ctypes.create_string_buffer(_CAP)
    nz = ctypes.c_uint64(0)
    m = len(moduli)
    mods = (ctypes.c_uint32 * max(m, 1))(*moduli)
    res = (ctypes.c_uint32 * max(m, 1))()
    rc = lib.godfrey_range(kind, n, index_begin, index_end, buf, _CAP, ctypes.byref(nz), mods, m, res)
    assert rc == 0, rc
    return int(buf.value), int(nz.value), [int(res[i]) for i in range(m)]


def chunk(kind: int, n: int, chunk_bits: int, c: int, moduli=()):
    """T(c): the sum over chunk c of the 2^chunk_bits chunks of the x_1 = +1 half:
    all indices v in [0, 2^{2n-1}) whose top chunk_bits bits equal c."""
    B = 2 * n - 1
    assert 0 <= chunk_bits <= B and 0 <= c < (1 << chunk_bits)
    w = 1 << (B - chunk_bits)
    return range_sum(kind, n, c * w, (c + 1) * w, moduli)


def total(kind: int, n: int, threads: int = 1):
    """Sigma_full over all 2^{2n} vectors (Lemma 2.1's sum before the division), and the non-zero
    term count.  `threads` > 1 only splits the index range into contiguous pieces summed afterwards
    with Python ints ("split ... into several independent sets and simply put the
    result together at the end")."""
    full = 1 << (2 * n)
    return _split(kind, n, 0, full, threads)


def _split(kind, n, lo, hi, threads):
    threads = max(1, min(threads, hi - lo))
    if threads == 1:
        s, nz, _ = range_sum(kind, n, lo, hi)
        return s, nz
    step = (hi - lo + threads - 1) // threads
    pieces = [(lo + i * step, min(hi, lo + (i + 1) * step)) for i in range(threads)]
    out = [None] * len(pieces)

    def work(i):
        out[i] = range_sum(kind, n, pieces[i][0], pieces[i][1])

    ts = [threading.Thread(target=work, args=(i,)) for i in range(len(pieces))]
    [t.start() for t in ts]
    [t.join() for t in ts]
    return sum(o[0] for o in out), sum(o[1] for o in out)


def count_distinct(kind: int, n: int, threads: int = 1) -> int:
    """D(n) = Sigma_full / 2^{2n}, asserting the division is exact (Lemma 2.1, reading A16)."""
    s, _ = total(kind, n, threads)
    q, r = divmod(s, 1 << (2 * n))
    assert r == 0, "Sigma_full not divisible by 2^{2n}"
    return q


def brute_count(kind: int, n: int) -> int:
    """Backtracking count, reflections distinct."""
    return int(_load().brute_count(kind, n))


def brute_list(kind: int, n: int, max_solutions: int = 4096):
    """All pairings as label sequences in position order (up to max_solutions)."""
    N = 2 * n
    arr = (ctypes.c_int * (N * max_solutions))()
    cnt = int(_load().brute_list(kind, n, arr, max_solutions))
    k = min(cnt, max_solutions)
    return cnt, [tuple(arr[i * N + j] for j in range(N)) for i in range(k)]

"""ctypes binding for include/pairings.h — same names, argument marshalling only."""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libpairings_b200.so")

SKOLEM, LANGFORD = 0, 1
VARIANT_AUTO, VARIANT_GENERIC, VARIANT_SWAR = 0, 1, 2
_CAP = 256

u32p = ctypes.POINTER(ctypes.c_uint32)
u64p = ctypes.POINTER(ctypes.c_uint64)


class LaunchOpts(ctypes.Structure):
    """struct pairings_launch_opts (include/pairings.h)."""
    _fields_ = [("variant", ctypes.c_int), ("gray_bits", ctypes.c_int), ("block_threads", ctypes.c_int),
                ("blocks_per_chunk", ctypes.c_int), ("nonzero_terms", ctypes.c_void_p)]


# int (*pairings_eval_fn)(void* ctx, int attempt, uint32_t* rows_out)
EVAL_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_uint32))


class PairingsError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__("%s: %s (code %d)" % (where, pairings_strerror(code), code))


_lib = None


def library_path() -> str:
    return _SO


def lib():
    """Loads libpairings_b200.so; fails loudly if it has not been built (python -m paper_1507_00315_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        raise ImportError("libpairings_b200.so is missing at %s — build it with "
                          "`python -m paper_1507_00315_b200.build` (there is no CPU fallback)" % _SO)
    L = ctypes.CDLL(_SO)
    i, u64, vp, cp = ctypes.c_int, ctypes.c_uint64, ctypes.c_void_p, ctypes.c_char_p
    optp = ctypes.POINTER(LaunchOpts)
    sigs = {
        "count_pairings": (i, [i, i, i, u64, u64, u32p, i, vp, vp]),
        "count_pairings_ex": (i, [i, i, i, u64, u64, u32p, i, vp, vp, optp]),
        "count_pairings_host": (i, [i, i, i, u64, u64, u32p, i, u32p, vp, optp]),
        "pairings_has_swar": (i, [i, i]),
        "pairings_query_geometry": (i, [i, i, i, u64, optp, ctypes.POINTER(i), ctypes.POINTER(i), ctypes.POINTER(i),
                                        ctypes.POINTER(i)]),
        "pairings_default_moduli": (i, [u32p, i]),
        "pairings_min_moduli": (i, [i, i]),
        "pairings_bound_moduli": (i, [i, i]),
        "pairings_partition": (ctypes.c_int64, [i, u64, u64p, i, u64p, ctypes.c_int64]),
        "pairings_rank_range": (i, [i, i, i, u64p, u64p]),
        "pairings_sum_rows": (i, [u32p, u64, u32p, i, u32p]),
        "pairings_journal_append": (i, [cp, i, i, i, u32p, i, u64, u64, u32p]),
        "pairings_journal_load": (ctypes.c_int64, [cp, i, i, i, u32p, i, u64p, ctypes.c_int64, u32p]),
        "pairings_run": (i, [i, i, i, u32p, i, u64, cp, ctypes.c_int64, vp, optp, u32p, u64p]),
        "pairings_run_ex": (i, [i, i, i, u32p, i, u64, cp, ctypes.c_int64, vp, optp, ctypes.c_uint, u32p, u64p, u64p, u64p]),
        "pairings_run_slice": (i, [i, i, i, u32p, i, u64, cp, ctypes.c_int64, vp, optp, ctypes.c_uint, u64, u64, u32p, u64p, u64p,
                                   u64p]),
        "pairings_journal_merge": (ctypes.c_int64, [ctypes.POINTER(cp), i, cp, i, i, i, u32p, i, u32p, u64p]),
        "pairings_journal_merge_mode": (ctypes.c_int64, [ctypes.POINTER(cp), i, cp, i, i, i, u32p, i, ctypes.c_uint, u32p, u64p,
                                                         u64p]),
        "pairings_mode_chunks": (i, [i, i, i, ctypes.c_uint, u64p]),
        "pairings_finish_total": (i, [i, i, i, ctypes.c_uint, u64, u32p, i, u32p]),
        "pairings_vote_rows": (i, [u32p, u32p, u32p, u64]),
        "pairings_duplicate_vote": (i, [EVAL_FN, vp, u64, u32p, ctypes.POINTER(i)]),
        "pairings_lemma24": (i, [i, i]),
        "pairings_reconstruct": (i, [i, i, u32p, i, u32p, cp, cp, ctypes.c_size_t]),
        "pairings_crt_signed": (i, [u32p, i, u32p, cp, ctypes.c_size_t]),
        "pairings_pt_run": (i, [i, i, ctypes.POINTER(ctypes.c_double), i, u64, u64, u64, u64, u64, vp, vp, vp, vp]),
        "pairings_pt_run_noalloc": (i, [i, i, ctypes.POINTER(ctypes.c_double), i, u64, u64, u64, u64, u64, vp, vp, vp, vp]),
        "pairings_pt_ladder": (i, [i, i, ctypes.c_double, u64, u64, u64, ctypes.POINTER(ctypes.c_double), i, vp]),
        "pairings_pt_counts": (i, [i, ctypes.c_double, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]),
        "pairings_pt_estimate": (i, [i, i, ctypes.POINTER(ctypes.c_double), i, u64p, ctypes.POINTER(ctypes.c_double),
                                     ctypes.POINTER(ctypes.c_double)]),
        "pairings_strerror": (cp, [i]),
        "pairings_build_info": (cp, []),
    }
    for name, (res, args) in sigs.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


def _u32(values: Sequence[int]):
    return (ctypes.c_uint32 * max(len(values), 1))(*values)


def _opts(opts: Optional[LaunchOpts]):
    return ctypes.byref(opts) if opts is not None else None


def _check(rc: int, where: str):
    if rc < 0:
        raise PairingsError(int(rc), where)
    return rc


def pairings_strerror(code: int) -> str:
    return lib().pairings_strerror(int(code)).decode()


def pairings_build_info() -> str:
    return lib().pairings_build_info().decode()


def pairings_has_swar(kind: int, n: int) -> bool:
    return bool(lib().pairings_has_swar(kind, n))


def pairings_query_geometry(kind, n, chunk_bits, n_chunks, opts: Optional[LaunchOpts] = None):
    """(variant, gray_bits, block_threads, blocks_per_chunk) of a count_pairings_ex call over n_chunks chunks."""
    v, g, t, b = ctypes.c_int(0), ctypes.c_int(0), ctypes.c_int(0), ctypes.c_int(0)
    _check(lib().pairings_query_geometry(kind, n, chunk_bits, n_chunks, _opts(opts), ctypes.byref(v), ctypes.byref(g),
                                         ctypes.byref(t), ctypes.byref(b)), "pairings_query_geometry")
    return int(v.value), int(g.value), int(t.value), int(b.value)


def count_pairings(kind, n, chunk_bits, chunk_begin, chunk_end, moduli, out_residues_ptr: int, stream: int = 0):
    """out_residues_ptr: DEVICE pointer (int, e.g. tensor.data_ptr()); stream: cudaStream_t as int."""
    m = _u32(moduli)
    _check(lib().count_pairings(kind, n, chunk_bits, chunk_begin, chunk_end, m, len(moduli),
                                ctypes.c_void_p(out_residues_ptr), ctypes.c_void_p(stream)), "count_pairings")


def count_pairings_ex(kind, n, chunk_bits, chunk_begin, chunk_end, moduli, out_residues_ptr: int, stream: int = 0,
                      opts: Optional[LaunchOpts] = None):
    m = _u32(moduli)
    _check(lib().count_pairings_ex(kind, n, chunk_bits, chunk_begin, chunk_end, m, len(moduli),
                                   ctypes.c_void_p(out_residues_ptr), ctypes.c_void_p(stream), _opts(opts)),
           "count_pairings_ex")


def count_pairings_host(kind, n, chunk_bits, chunk_begin, chunk_end, moduli, stream: int = 0,
                        opts: Optional[LaunchOpts] = None, out=None):
    """Returns the rows as a list of lists (or fills `out`, a ctypes uint32 array, and returns it)."""
    m = _u32(moduli)
    rows = chunk_end - chunk_begin
    ret_list = out is None
    if out is None:
        out = (ctypes.c_uint32 * max(rows * len(moduli), 1))()
    _check(lib().count_pairings_host(kind, n, chunk_bits, chunk_begin, chunk_end, m, len(moduli), out,
                                     ctypes.c_void_p(stream), _opts(opts)), "count_pairings_host")
    if not ret_list:
        return out
    k = len(moduli)
    return [[int(out[r * k + j]) for j in range(k)] for r in range(rows)]


def pairings_default_moduli(count: int):
    out = (ctypes.c_uint32 * max(count, 1))()
    _check(lib().pairings_default_moduli(out, count), "pairings_default_moduli")
    return [int(out[j]) for j in range(count)]


def pairings_min_moduli(kind: int, n: int) -> int:
    return _check(lib().pairings_min_moduli(kind, n), "pairings_min_moduli")


def pairings_bound_moduli(kind: int, n: int) -> int:
    return _check(lib().pairings_bound_moduli(kind, n), "pairings_bound_moduli")


def pairings_partition(chunk_bits: int, max_chunks: int, done=()):
    flat = [v for r in done for v in r]
    d = (ctypes.c_uint64 * max(len(flat), 1))(*flat)
    need = _check(lib().pairings_partition(chunk_bits, max_chunks, d, len(done), None, 0), "pairings_partition")
    out = (ctypes.c_uint64 * max(2 * need, 1))()
    _check(lib().pairings_partition(chunk_bits, max_chunks, d, len(done), out, need), "pairings_partition")
    return [(int(out[2 * j]), int(out[2 * j + 1])) for j in range(need)]


def pairings_rank_range(chunk_bits: int, rank: int, world: int):
    b, e = ctypes.c_uint64(0), ctypes.c_uint64(0)
    _check(lib().pairings_rank_range(chunk_bits, rank, world, ctypes.byref(b), ctypes.byref(e)), "pairings_rank_range")
    return int(b.value), int(e.value)


def pairings_sum_rows(rows, moduli, total=None):
    """rows: list of rows or a flat ctypes uint32 array (then pass n_rows via len(rows)//len(moduli))."""
    k = len(moduli)
    if isinstance(rows, ctypes.Array):
        flat, n_rows = rows, len(rows) // k
    else:
        vals = [v for r in rows for v in r]
        flat, n_rows = _u32(vals), len(rows)
    t = _u32(list(total) if total is not None else [0] * k)
    _check(lib().pairings_sum_rows(flat, n_rows, _u32(moduli), k, t), "pairings_sum_rows")
    return [int(t[j]) for j in range(k)]


def pairings_journal_append(path, kind, n, chunk_bits, moduli, chunk_begin, chunk_end, row_sum):
    _check(lib().pairings_journal_append(os.fsencode(path), kind, n, chunk_bits, _u32(moduli), len(moduli),
                                         chunk_begin, chunk_end, _u32(row_sum)), "pairings_journal_append")


def pairings_journal_load(path, kind, n, chunk_bits, moduli):
    k = len(moduli)
    t = _u32([0] * k)
    need = _check(lib().pairings_journal_load(os.fsencode(path), kind, n, chunk_bits, _u32(moduli), k, None, 0, t),
                  "pairings_journal_load")
    out = (ctypes.c_uint64 * max(2 * need, 1))()
    _check(lib().pairings_journal_load(os.fsencode(path), kind, n, chunk_bits, _u32(moduli), k, out, need, t),
           "pairings_journal_load")
    return [(int(out[2 * j]), int(out[2 * j + 1])) for j in range(need)], [int(t[j]) for j in range(k)]


def pairings_run(kind, n, chunk_bits, moduli, chunks_per_call, journal_path=None, max_calls=0, stream: int = 0,
                 opts: Optional[LaunchOpts] = None):
    """Whole-job host driver.  Returns (total residues, chunks done)."""
    k = len(moduli)
    t = _u32([0] * k)
    done = ctypes.c_uint64(0)
    jp = os.fsencode(journal_path) if journal_path is not None else None
    _check(lib().pairings_run(kind, n, chunk_bits, _u32(moduli), k, chunks_per_call, jp, max_calls,
                              ctypes.c_void_p(stream), _opts(opts), t, ctypes.byref(done)), "pairings_run")
    return [int(t[j]) for j in range(k)], int(done.value)


RUN_LEMMA24, RUN_DUPLICATE, RUN_AUDIT = 1, 2, 4


def pairings_lemma24(kind: int, n: int) -> int:
    """1: term(x^) = term(x) (pairings exist); 0: term(x^) = -term(x) (H = 0).  Lemma 2.4."""
    return _check(lib().pairings_lemma24(kind, n), "pairings_lemma24")


def pairings_run_ex(kind, n, chunk_bits, moduli, chunks_per_call, journal_path=None, max_calls=0, stream: int = 0,
                    opts: Optional[LaunchOpts] = None, flags: int = 0):
    """Whole-job host driver with flags.  Returns (total residues, chunks done, chunks needed); the number of
    duplicate-run mismatches of the last call is kept in pairings_run_ex.last_mismatches."""
    k = len(moduli)
    t = _u32([0] * k)
    done, needed, mism = ctypes.c_uint64(0), ctypes.c_uint64(0), ctypes.c_uint64(0)
    jp = os.fsencode(journal_path) if journal_path is not None else None
    _check(lib().pairings_run_ex(kind, n, chunk_bits, _u32(moduli), k, chunks_per_call, jp, max_calls,
                                 ctypes.c_void_p(stream), _opts(opts), flags, t, ctypes.byref(done),
                                 ctypes.byref(needed), ctypes.byref(mism)), "pairings_run_ex")
    pairings_run_ex.last_mismatches = int(mism.value)
    return [int(t[j]) for j in range(k)], int(done.value), int(needed.value)


def pairings_run_slice(kind, n, chunk_bits, moduli, chunks_per_call, slice_begin, slice_end, journal_path=None, max_calls=0,
                       stream: int = 0, opts: Optional[LaunchOpts] = None, flags: int = 0):
    """One job of a chunk farm: pairings_run_ex over the chunks of [slice_begin, slice_end) only.  Returns (summed
    rows of the slice, chunks done, chunks this slice needs); mismatches in pairings_run_slice.last_mismatches."""
    k = len(moduli)
    t = _u32([0] * k)
    done, needed, mism = ctypes.c_uint64(0), ctypes.c_uint64(0), ctypes.c_uint64(0)
    jp = os.fsencode(journal_path) if journal_path is not None else None
    _check(lib().pairings_run_slice(kind, n, chunk_bits, _u32(moduli), k, chunks_per_call, jp, max_calls,
                                    ctypes.c_void_p(stream), _opts(opts), flags, slice_begin, slice_end, t,
                                    ctypes.byref(done), ctypes.byref(needed), ctypes.byref(mism)), "pairings_run_slice")
    pairings_run_slice.last_mismatches = int(mism.value)
    return [int(t[j]) for j in range(k)], int(done.value), int(needed.value)


def pairings_journal_merge(paths, kind, n, chunk_bits, moduli, out_path=None):
    """Adds up the journals of several jobs.  Returns (ranges, total residues, chunks covered)."""
    k = len(moduli)
    arr = (ctypes.c_char_p * len(paths))(*[os.fsencode(p) for p in paths])
    t = _u32([0] * k)
    cov = ctypes.c_uint64(0)
    nr = _check(lib().pairings_journal_merge(arr, len(paths), os.fsencode(out_path) if out_path is not None else None,
                                             kind, n, chunk_bits, _u32(moduli), k, t, ctypes.byref(cov)),
                "pairings_journal_merge")
    return int(nr), [int(t[j]) for j in range(k)], int(cov.value)


def pairings_journal_merge_mode(paths, kind, n, chunk_bits, moduli, flags: int = 0, out_path=None):
    """pairings_journal_merge for a job mode (RUN_* flags): ranges outside the chunks that mode evaluates are refused.
    Returns (ranges, raw total residues, chunks covered, chunks needed); finish with pairings_finish_total."""
    arr = (ctypes.c_char_p * len(paths))(*[os.fsencode(p) for p in paths])
    total = (ctypes.c_uint32 * len(moduli))()
    cov, need = ctypes.c_uint64(0), ctypes.c_uint64(0)
    nr = _check(lib().pairings_journal_merge_mode(arr, len(paths), os.fsencode(out_path) if out_path else None, kind, n,
                                                  chunk_bits, _u32(moduli), len(moduli), flags, total, ctypes.byref(cov),
                                                  ctypes.byref(need)), "pairings_journal_merge_mode")
    return nr, [int(v) for v in total], int(cov.value), int(need.value)


def pairings_mode_chunks(kind, n, chunk_bits, flags: int = 0):
    """(chunks a whole job evaluates in this mode — always the range [0, needed) —, factor 1 / 2 / 0 that turns
    their sum into H).  Lemma 2.4."""
    need = ctypes.c_uint64(0)
    f = _check(lib().pairings_mode_chunks(kind, n, chunk_bits, flags, ctypes.byref(need)), "pairings_mode_chunks")
    return int(need.value), f


def pairings_finish_total(kind, n, chunk_bits, flags, chunks_covered, moduli, total):
    """(complete?, total): when chunks_covered is the mode's whole chunk count, `total` (raw row sum) times the
    mode's factor = H mod p_i, ready for pairings_reconstruct; otherwise (False, total unchanged)."""
    t = _u32(total)
    rc = _check(lib().pairings_finish_total(kind, n, chunk_bits, flags, chunks_covered, _u32(moduli), len(moduli), t),
                "pairings_finish_total")
    return bool(rc), [int(v) for v in t]


def pairings_vote_rows(a, b, c=None) -> int:
    """0: a stands, 1: b stands, 3: a != b and no third run given; raises PairingsError(ECHECK) if no two agree."""
    return _check(lib().pairings_vote_rows(_u32(a), _u32(b), _u32(c) if c is not None else None, len(a)),
                  "pairings_vote_rows")


def pairings_duplicate_vote(evaluate, n_words: int):
    """evaluate(attempt) -> list of n_words ints (or a negative error code).  Returns (rows, mismatch).
    An exception raised by evaluate, or a row of the wrong length, stops the vote (the C side sees PAIRINGS_ECHECK, so
    two failed attempts can never 'agree' on unfilled rows) and is re-raised here."""
    failure = []

    def thunk(_ctx, attempt, out):
        try:                                      # ctypes would swallow the exception and hand 0 (= success) to C
            r = evaluate(int(attempt))
            if isinstance(r, int):
                return r if r < 0 else -7         # a code is an error; 0 or positive without rows is one too
            r = list(r)
            if len(r) != n_words:
                raise ValueError("evaluate(%d) returned %d words, expected %d" % (attempt, len(r), n_words))
            for j, v in enumerate(r):
                out[j] = v
            return 0
        except BaseException as exc:              # noqa: BLE001 — re-raised after the C call returns
            failure.append(exc)
            return -7
    cb = EVAL_FN(thunk)
    rows = (ctypes.c_uint32 * max(n_words, 1))()
    mm = ctypes.c_int(0)
    rc = lib().pairings_duplicate_vote(cb, None, n_words, rows, ctypes.byref(mm))
    if failure:
        raise failure[0]
    _check(rc, "pairings_duplicate_vote")
    return [int(rows[j]) for j in range(n_words)], int(mm.value)


def pairings_reconstruct(kind, n, moduli, total_residues):
    """Returns (D, S) = (reflections distinct, reflections identified) as Python ints."""
    a, b = ctypes.create_string_buffer(_CAP), ctypes.create_string_buffer(_CAP)
    _check(lib().pairings_reconstruct(kind, n, _u32(moduli), len(moduli), _u32(total_residues), a, b, _CAP),
           "pairings_reconstruct")
    return int(a.value), int(b.value)


def pairings_crt_signed(moduli, residues) -> int:
    a = ctypes.create_string_buffer(_CAP)
    _check(lib().pairings_crt_signed(_u32(moduli), len(moduli), _u32(residues), a, _CAP), "pairings_crt_signed")
    return int(a.value)


def pairings_pt_run(kind, n, betas, replica_begin, replica_end, iterations, burn_in, seed, hist_dev_ptr: int,
                    moves_dev_ptr: int, swaps_dev_ptr: int, stream: int = 0):
    """Approximate counter (Algorithm 2): ADDS to the DEVICE counters hist (levels x (2n+1)
    uint64), moves and swaps (levels uint64 each)."""
    b = (ctypes.c_double * len(betas))(*betas)
    _check(lib().pairings_pt_run(kind, n, b, len(betas), replica_begin, replica_end, iterations, burn_in, seed,
                                 ctypes.c_void_p(hist_dev_ptr), ctypes.c_void_p(moves_dev_ptr),
                                 ctypes.c_void_p(swaps_dev_ptr), ctypes.c_void_p(stream)), "pairings_pt_run")


def pairings_pt_run_noalloc(kind, n, betas, replica_begin, replica_end, iterations, burn_in, seed, hist_dev_ptr: int,
                            moves_dev_ptr: int, swaps_dev_ptr: int, stream: int = 0):
    """pairings_pt_run without any device allocation, for programs that cannot call cudaMalloc (all memory already
    in their own arena, a latency budget, or a host application that forbids it): the kernel's threshold table sits
    in a fixed 16 KiB array inside the library.  Same arguments and counters; n_levels * (2n + 3) must be <= 2048
    (PairingsError with code -12 otherwise).  All calls on one device share that array, so calls whose GPU work may
    overlap race; the first call on a device does a one-off address look-up and should precede any stream capture."""
    b = (ctypes.c_double * len(betas))(*betas)
    _check(lib().pairings_pt_run_noalloc(kind, n, b, len(betas), replica_begin, replica_end, iterations, burn_in, seed,
                                         ctypes.c_void_p(hist_dev_ptr), ctypes.c_void_p(moves_dev_ptr),
                                         ctypes.c_void_p(swaps_dev_ptr), ctypes.c_void_p(stream)),
           "pairings_pt_run_noalloc")


def pairings_pt_ladder(kind, n, target_exchange=0.55, pilot_replicas=256, pilot_iterations=1 << 14, seed=1,
                       cap_levels=32, stream: int = 0):
    """Inverse-temperature ladder with the given predicted exchange acceptance.  Returns the betas."""
    out = (ctypes.c_double * cap_levels)()
    m = _check(lib().pairings_pt_ladder(kind, n, target_exchange, pilot_replicas, pilot_iterations, seed, out,
                                        cap_levels, ctypes.c_void_p(stream)), "pairings_pt_ladder")
    return [float(out[j]) for j in range(m)]


def pairings_pt_estimate(kind, n, betas, hist):
    """hist: levels x (2n+1) counts.  Returns (ratios per level, log of the estimated reflections-distinct count)."""
    M = len(betas)
    b = (ctypes.c_double * M)(*betas)
    flat = (ctypes.c_uint64 * (M * (2 * n + 1)))(*[int(v) for row in hist for v in row])
    r = (ctypes.c_double * M)()
    lz = ctypes.c_double(0.0)
    _check(lib().pairings_pt_estimate(kind, n, b, M, flat, r, ctypes.byref(lz)), "pairings_pt_estimate")
    return [float(v) for v in r], float(lz.value)


def pairings_pt_counts(n: int, log_distinct: float):
    """(distinct, identified) estimates from pairings_pt_estimate's logarithm (Table 6 caption)."""
    d, s_ = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(lib().pairings_pt_counts(n, log_distinct, ctypes.byref(d), ctypes.byref(s_)), "pairings_pt_counts")
    return float(d.value), float(s_.value)


def approx_count(kind: int, n: int, replicas: int = 1 << 12, iterations: int = 1 << 16, burn_in: Optional[int] = None,
                 seed: int = 150700315, betas=None, target_exchange: float = 0.55, device_alloc=None):
    """Convenience: the approximate counter end to end (§3) — ladder (unless given), one pairings_pt_run,
    estimate.  Needs torch for the device counters unless `device_alloc(n_uint64) -> (ptr, read)` is given.
    Returns dict(identified, distinct, betas, ratios, moves, swaps, samples)."""
    import torch
    if betas is None:
        betas = pairings_pt_ladder(kind, n, target_exchange, 256, 1 << (14 if n <= 16 else 18), seed ^ 0x5bd1e995)
    if burn_in is None:
        burn_in = iterations // 2
    M, N = len(betas), 2 * n
    hist = torch.zeros((M, N + 1), dtype=torch.int64, device="cuda")
    mv = torch.zeros(M, dtype=torch.int64, device="cuda")
    sw = torch.zeros(M, dtype=torch.int64, device="cuda")
    done = 0
    while done < replicas:                          # at most 2^30 replicas and 2^25 iterations per call
        take = min(replicas - done, 1 << 20)
        pairings_pt_run(kind, n, betas, done, done + take, iterations, burn_in, seed, hist.data_ptr(), mv.data_ptr(),
                        sw.data_ptr(), torch.cuda.current_stream().cuda_stream)
        done += take
    torch.cuda.synchronize()
    h = hist.cpu().tolist()
    ratios, logz = pairings_pt_estimate(kind, n, betas, h)
    distinct, identified = pairings_pt_counts(n, logz)
    return dict(distinct=distinct, identified=identified, betas=betas, ratios=ratios,
                moves=mv.cpu().tolist(), swaps=sw.cpu().tolist(), samples=replicas * (iterations - burn_in))


def default_chunk_bits(n: int) -> int:
    """2^23 sign vectors per chunk (one block of 256 threads x 2^15 terms), at most 2^20 chunks."""
    return max(0, min(2 * n - 1 - 23, 20))


def default_chunks_per_call(n: int, chunk_bits: int) -> int:
    """About 2^41 sign vectors per kernel call (a few seconds): few launches, journal lines, D2H copies, and a
    last partly filled wave of blocks that is short against the call."""
    return 1 << max(0, min(chunk_bits, 41 - (2 * n - 1 - chunk_bits)))


def count(kind: int, n: int, chunk_bits: Optional[int] = None, n_moduli: Optional[int] = None,
          chunks_per_call: Optional[int] = None, journal_path=None, opts: Optional[LaunchOpts] = None,
          lemma24: bool = False, duplicate: bool = False, tight_moduli: bool = False):
    """Convenience: the whole path for (kind, n) -> (D, S).  Calls only the C ABI."""
    if n_moduli is None:      # §8(f) NEXT #2: the tight bound 2^{2n-1} prod(2n-d_k) instead of north_star's (2n)^n 2^{2n}
        n_moduli = (pairings_min_moduli(kind, n) if tight_moduli else pairings_bound_moduli(kind, n)) + 1
    moduli = pairings_default_moduli(n_moduli)
    if chunk_bits is None:
        chunk_bits = default_chunk_bits(n)
    if chunks_per_call is None:
        chunks_per_call = default_chunks_per_call(n, chunk_bits)
    total, done, needed = pairings_run_ex(kind, n, chunk_bits, moduli, chunks_per_call, journal_path, 0, 0, opts,
                                          (RUN_LEMMA24 if lemma24 else 0) | (RUN_DUPLICATE if duplicate else 0))
    assert done == needed
    return pairings_reconstruct(kind, n, moduli, total)

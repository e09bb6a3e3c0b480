"""Command line: the whole path for one (kind, n), with journal / resume.

    python -m paper_1507_00315_b200 S 24 [--chunk-bits 20] [--moduli 9] [--chunks-per-call 8192]
                                         [--journal FILE] [--max-calls K] [--lemma24] [--json]

Prints D(n) (reflections distinct) and S(n) / L(n) (reflections identified, the paper's numbers,
PAPER.md:63) and the wall time.  Calls only the C ABI (pairings_run + pairings_reconstruct); an
interrupted run (--max-calls, or a crash) continues from the journal when started again.
"""
from __future__ import annotations

import argparse
import json
import sys
import time

from . import api


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(prog="python -m paper_1507_00315_b200")
    ap.add_argument("kind", choices=["S", "L", "s", "l"], help="S = Skolem (d_k = k), L = Langford (d_k = k+1)")
    ap.add_argument("n", type=int)
    ap.add_argument("--chunk-bits", type=int, default=None)
    ap.add_argument("--moduli", type=int, default=None, help="CRT primes + 1 check prime (default: north_star bound + 1)")
    ap.add_argument("--chunks-per-call", type=int, default=None)
    ap.add_argument("--lemma24", action="store_true",
                    help="symmetry 3 (Lemma 2.4, PAPER.md:215-249): evaluate only the x_2 = +1 half and double it")
    ap.add_argument("--duplicate", action="store_true",
                    help="PAPER.md:99: evaluate every chunk range twice (other launch geometry), third run on mismatch")
    ap.add_argument("--tight-moduli", action="store_true",
                    help="size the prime set from 2^(2n-1) prod(2n-d_k) instead of (2n)^n 2^(2n)")
    ap.add_argument("--approx", action="store_true",
                    help="approximate count by parallel tempering (PAPER.md section 3) instead of the exact count")
    ap.add_argument("--replicas", type=int, default=1 << 12)
    ap.add_argument("--iterations", type=int, default=None, help="per replica (default 2^16, 2^21 for n >= 20, 2^23 for n >= 24)")
    ap.add_argument("--journal", default=None)
    ap.add_argument("--max-calls", type=int, default=0)
    ap.add_argument("--json", action="store_true")
    a = ap.parse_args(argv)

    kind = api.SKOLEM if a.kind.upper() == "S" else api.LANGFORD
    n = a.n
    if a.approx:
        its = a.iterations if a.iterations is not None else (1 << 16 if n < 20 else (1 << 21 if n < 24 else 1 << 23))
        t0 = time.perf_counter()
        r = api.approx_count(kind, n, a.replicas, its)
        r["seconds"] = time.perf_counter() - t0
        if a.json:
            print(json.dumps(r))
        else:
            print("%s(%d) ~ %.6g (reflections identified; %d levels, %.3g samples per level, %.2f s)" %
                  (a.kind.upper(), n, r["identified"], len(r["betas"]), r["samples"], r["seconds"]))
        return 0
    m = a.moduli if a.moduli is not None else \
        (api.pairings_min_moduli(kind, n) if a.tight_moduli else api.pairings_bound_moduli(kind, n)) + 1
    moduli = api.pairings_default_moduli(m)
    C = a.chunk_bits if a.chunk_bits is not None else api.default_chunk_bits(n)
    per_call = a.chunks_per_call if a.chunks_per_call is not None else api.default_chunks_per_call(n, C)
    ti = time.perf_counter()
    api.count_pairings_host(api.LANGFORD, 3, 0, 0, 1, moduli[:1])      # CUDA context + module load, outside the timing
    init_s = time.perf_counter() - ti
    t0 = time.perf_counter()
    total, done, needed = api.pairings_run_ex(kind, n, C, moduli, per_call, a.journal, a.max_calls, 0, None,
                                              (api.RUN_LEMMA24 if a.lemma24 else 0) |
                                              (api.RUN_DUPLICATE if a.duplicate else 0))
    dt = time.perf_counter() - t0
    res = dict(kind=a.kind.upper(), n=n, chunk_bits=C, moduli=moduli, chunks_done=done, chunks_needed=needed,
               chunks=1 << C, lemma24=bool(a.lemma24), duplicate=bool(a.duplicate),
               duplicate_mismatches=api.pairings_run_ex.last_mismatches, seconds=dt, init_seconds=init_s, total_residues=total)
    if done == needed:
        D, S = api.pairings_reconstruct(kind, n, moduli, total)
        evaluated = needed << (2 * n - 1 - C)
        res.update(distinct=D, identified=S, terms_evaluated=evaluated, terms_per_s=evaluated / dt if dt > 0 else None)
    if a.json:
        print(json.dumps(res))
    elif done == needed:
        print("%s(%d): reflections identified %d, distinct %d  (%.2f s in this call, %d chunks)" %
              (res["kind"], n, res["identified"], res["distinct"], dt, done))
    else:
        print("%s(%d): %d of %d chunks done (%.2f s in this call); run again to continue" %
              (res["kind"], n, done, needed, dt))
    return 0


if __name__ == "__main__":
    sys.exit(main())

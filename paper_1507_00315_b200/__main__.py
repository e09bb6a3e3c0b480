"""Command line: the whole path for one (kind, n), with journal / resume.

    python -m paper_1507_00315_b200 S 24 [--chunk-bits 20] [--moduli 9] [--chunks-per-call 8192]
                                         [--journal FILE] [--max-calls K] [--lemma24] [--duplicate] [--audit] [--json]

Prints D(n) (reflections distinct) and S(n) / L(n) (reflections identified, the paper's numbers,
PAPER.md:63) and the wall time.  Calls only the C ABI (pairings_run_slice + pairings_reconstruct); an
interrupted run (--max-calls, or a crash) continues from the journal when started again.

Chunk farm ("split ... into several independent sets and simply put the result together at the end";
PAPER.md:257: S(25) as 4 GPU jobs, L(27) 64, n = 28 256, S(29) 1024) — one job per GPU, any machine, any time:

    CUDA_VISIBLE_DEVICES=r python -m paper_1507_00315_b200 S 25 --lemma24 --rank r --world 4 --journal j_r.txt    # r = 0..3
    python -m paper_1507_00315_b200 S 25 --lemma24 --merge j_0.txt j_1.txt j_2.txt j_3.txt [--journal merged.txt]

A job evaluates the slice pairings_rank_range deals to its rank (of the chunks this mode evaluates) into its own
journal; --merge adds the journals up (pairings_journal_merge: overlapping or foreign journals are refused),
applies the symmetry factor and reconstructs.  Jobs and merge must be given the same kind, n, --chunk-bits,
--moduli / --tight-moduli and --lemma24.
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
    ap.add_argument("--audit", action="store_true",
                    help="re-evaluate two chunks of every range with the generic kernel (an independent implementation) and compare")
    ap.add_argument("--rank", type=int, default=0, help="chunk farm: this job's rank (with --world)")
    ap.add_argument("--world", type=int, default=1, help="chunk farm: number of jobs the chunks are dealt to")
    ap.add_argument("--merge", nargs="+", default=None, metavar="JOURNAL",
                    help="chunk farm: add up the jobs' journals and reconstruct (no GPU needed)")
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
    flags = (api.RUN_LEMMA24 if a.lemma24 else 0) | (api.RUN_DUPLICATE if a.duplicate else 0) | (api.RUN_AUDIT if a.audit else 0)
    # chunks [0, job_chunks) are what this mode evaluates; Lemma 2.4's rule lives behind the ABI (pairings_mode_chunks,
    # pairings_finish_total), the command line never applies a factor of its own
    job_chunks, _factor = api.pairings_mode_chunks(kind, n, C, flags)

    if a.merge is not None:                                       # put the jobs' results together (host only)
        t0 = time.perf_counter()
        if job_chunks == 0:
            ranges, total, covered = 0, [0] * m, 0
        else:
            ranges, total, covered, _needed = api.pairings_journal_merge_mode(a.merge, kind, n, C, moduli, flags, a.journal)
        res = dict(kind=a.kind.upper(), n=n, chunk_bits=C, moduli=moduli, merged=list(a.merge), ranges=ranges,
                   chunks_done=covered, chunks_needed=job_chunks, lemma24=bool(a.lemma24), total_residues=total,
                   seconds=time.perf_counter() - t0)
        complete, total = api.pairings_finish_total(kind, n, C, flags, covered, moduli, total)
        if complete:
            D, S = api.pairings_reconstruct(kind, n, moduli, total)
            res.update(distinct=D, identified=S, total_residues=total)
        if a.json:
            print(json.dumps(res))
        elif complete:
            print("%s(%d): reflections identified %d, distinct %d  (%d journals, %d ranges)" %
                  (res["kind"], n, res["identified"], res["distinct"], len(a.merge), ranges))
        else:
            print("%s(%d): the journals cover %d of %d chunks; the count needs all of them" % (res["kind"], n, covered, job_chunks))
        return 0 if complete else 3

    if not 0 <= a.rank < a.world:
        ap.error("--rank must be in [0, --world)")
    # this job's slice of the chunks the mode evaluates: [0, 2^C), or its x_2 = +1 half [0, 2^(C-1))
    if job_chunks == 0:
        sb = se = 0
    elif a.world == 1:
        sb, se = 0, job_chunks
    else:
        sb, se = api.pairings_rank_range(job_chunks.bit_length() - 1, a.rank, a.world)     # job_chunks is a power of two
    ti = time.perf_counter()
    api.count_pairings_host(api.LANGFORD, 3, 0, 0, 1, moduli[:1])      # CUDA context + module load, outside the timing
    init_s = time.perf_counter() - ti
    t0 = time.perf_counter()
    total, done, needed = api.pairings_run_slice(kind, n, C, moduli, per_call, sb, se, a.journal, a.max_calls, 0, None, flags)
    dt = time.perf_counter() - t0
    res = dict(kind=a.kind.upper(), n=n, chunk_bits=C, moduli=moduli, chunks_done=done, chunks_needed=needed,
               chunks=1 << C, slice=[sb, se], rank=a.rank, world=a.world, lemma24=bool(a.lemma24), duplicate=bool(a.duplicate),
               audit=bool(a.audit), duplicate_mismatches=api.pairings_run_slice.last_mismatches, seconds=dt, init_seconds=init_s,
               total_residues=total)
    if res["duplicate_mismatches"]:                               # a vote was needed: the count stands, the hardware is suspect
        sys.stderr.write("warning: %d chunk range(s) had disagreeing runs and were settled by a vote (PAPER.md:99); "
                         "check this GPU\n" % res["duplicate_mismatches"])
    evaluated = needed << (2 * n - 1 - C)
    res.update(terms_evaluated=evaluated, terms_per_s=evaluated / dt if dt > 0 and done == needed else None)
    whole = False
    if a.world == 1:                                              # a slice run alone: finished like merged journals
        whole, total = api.pairings_finish_total(kind, n, C, flags, done, moduli, total)
    if whole:
        D, S = api.pairings_reconstruct(kind, n, moduli, total)
        res.update(distinct=D, identified=S, total_residues=total)
    if a.json:
        print(json.dumps(res))
    elif whole:
        print("%s(%d): reflections identified %d, distinct %d  (%.2f s in this call, %d chunks)" %
              (res["kind"], n, res["identified"], res["distinct"], dt, done))
    elif done == needed:
        print("%s(%d): job %d of %d done, chunks [%d, %d) (%.2f s in this call); put the journals together with --merge" %
              (res["kind"], n, a.rank, a.world, sb, se, dt))
    else:
        print("%s(%d): %d of %d chunks done (%.2f s in this call); run again to continue" %
              (res["kind"], n, done, needed, dt))
    return 0


if __name__ == "__main__":
    sys.exit(main())

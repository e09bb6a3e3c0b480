"""CPU-only tests of the C-ABI library: symbol export, argument validation (before any launch),
moduli, partitioner, journal, row sums and CRT (against Python integers).  No compute calls."""
import ctypes
import os
import random
import re

import pytest

import paper_1507_00315_b200 as pb
from paper_1507_00315_b200 import build as pbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="session", autouse=True)
def built():
    pbuild.build()
    return pb.lib()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "pairings.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = re.findall(r"\b(count_pairings\w*|pairings_\w+)\s*\(", text)
    return sorted(set(names))


def test_library_exports_every_declared_symbol(built):
    syms = declared_symbols()
    assert "count_pairings" in syms and "pairings_reconstruct" in syms and len(syms) >= 15
    for s in syms:
        assert hasattr(built, s), s


def test_strerror_and_build_info():
    assert pb.pairings_strerror(0) == "ok"
    for code in range(-12, 0):
        assert pb.pairings_strerror(code) != "unknown error code"
    assert "sm_100a" in pb.pairings_build_info()


def _is_prime(v):
    if v < 2:
        return False
    i = 2
    while i * i <= v:
        if v % i == 0:
            return False
        i += 1
    return True


def test_default_moduli_are_the_largest_primes_below_2_31():
    # reading A7: regenerated here by trial division, not copied
    want, v = [], (1 << 31) - 1
    while len(want) < 9:
        if _is_prime(v):
            want.append(v)
        v -= 2
    assert pb.pairings_default_moduli(9) == want
    assert want[0] == 2147483647


def test_min_moduli_matches_bound():
    for kind in (0, 1):
        for n in range(2, 33):
            bound = 2 * (1 << (2 * n - 1))
            for k in range(1, n + 1):
                bound *= 2 * n - (k if kind == 0 else k + 1)
            primes = pb.pairings_default_moduli(16)
            M, m = 1, 0
            while M <= bound:
                M *= primes[m]
                m += 1
            assert pb.pairings_min_moduli(kind, n) == m
            assert pb.pairings_bound_moduli(kind, n) >= m
    # BASELINE configs use 3,3,5,6,8 CRT primes: all at least the minimum
    for (kind, n, m) in ((1, 12, 3), (0, 13, 3), (0, 16, 5), (1, 16, 5), (1, 20, 6), (0, 21, 6), (0, 24, 8)):
        assert pb.pairings_min_moduli(kind, n) <= m


def test_argument_validation_happens_before_any_launch():
    good = pb.pairings_default_moduli(4)
    E = pb.PairingsError

    def code(fn):
        with pytest.raises(E) as ei:
            fn()
        return ei.value.code

    dummy = 0x1000  # never dereferenced: validation fails first
    assert code(lambda: pb.count_pairings(2, 12, 6, 0, 1, good, dummy)) == -1
    assert code(lambda: pb.count_pairings(0, 1, 0, 0, 1, good, dummy)) == -2
    assert code(lambda: pb.count_pairings(0, 33, 6, 0, 1, good, dummy)) == -2
    assert code(lambda: pb.count_pairings(0, 12, 24, 0, 1, good, dummy)) == -3
    assert code(lambda: pb.count_pairings(0, 12, -1, 0, 1, good, dummy)) == -3
    assert code(lambda: pb.count_pairings(0, 12, 6, 5, 4, good, dummy)) == -3
    assert code(lambda: pb.count_pairings(0, 12, 6, 0, 65, good, dummy)) == -3
    assert code(lambda: pb.count_pairings(0, 12, 6, 0, 1, [good[0], good[0]], dummy)) == -4
    assert code(lambda: pb.count_pairings(0, 12, 6, 0, 1, [2147483646], dummy)) == -4
    assert code(lambda: pb.count_pairings(0, 12, 6, 0, 1, [1073741789], dummy)) == -4   # < 2^30
    assert code(lambda: pb.count_pairings(0, 12, 6, 0, 1, [], dummy)) == -4
    assert code(lambda: pb.count_pairings(0, 12, 6, 0, 1, good, 0)) == -5
    assert code(lambda: pb.count_pairings_ex(0, 12, 6, 0, 1, good, dummy, 0, pb.LaunchOpts(variant=7))) == -10
    assert code(lambda: pb.count_pairings_ex(0, 12, 6, 0, 1, good, dummy, 0, pb.LaunchOpts(gray_bits=40))) == -10
    assert code(lambda: pb.count_pairings_ex(0, 12, 6, 0, 1, good, dummy, 0, pb.LaunchOpts(block_threads=48))) == -10
    assert code(lambda: pb.count_pairings_ex(0, 12, 6, 0, 1, good, dummy, 0, pb.LaunchOpts(blocks_per_chunk=3))) == -10
    # empty range: legal, nothing enqueued, no CUDA needed
    pb.count_pairings(0, 12, 6, 3, 3, good, 0)


def test_partition_covers_exactly_the_missing_chunks():
    rng = random.Random(150700315)
    for _ in range(200):
        C = rng.randrange(0, 9)
        total = 1 << C
        done = []
        for _ in range(rng.randrange(0, 5)):
            b = rng.randrange(0, total + 1)
            e = rng.randrange(b, total + 1)
            done.append((b, e))
        maxc = rng.randrange(1, 40)
        ranges = pb.pairings_partition(C, maxc, done)
        covered = set()
        for b, e in done:
            covered |= set(range(b, e))
        got = []
        for b, e in ranges:
            assert 0 < e - b <= maxc
            got += list(range(b, e))
        assert got == sorted(set(range(total)) - covered)


def test_rank_ranges_tile_the_chunk_space():
    for C in (0, 3, 16, 20):
        for world in (1, 2, 3, 4, 8):
            cur = 0
            sizes = []
            for r in range(world):
                b, e = pb.pairings_rank_range(C, r, world)
                assert b == cur and e >= b
                sizes.append(e - b)
                cur = e
            assert cur == 1 << C and max(sizes) - min(sizes) <= 1


def test_sum_rows_mod_p():
    rng = random.Random(1)
    moduli = pb.pairings_default_moduli(5)
    rows = [[rng.randrange(p) for p in moduli] for _ in range(1000)]
    start = [rng.randrange(p) for p in moduli]
    got = pb.pairings_sum_rows(rows, moduli, start)
    assert got == [(start[j] + sum(r[j] for r in rows)) % p for j, p in enumerate(moduli)]


def test_crt_roundtrip_random_big_integers():
    rng = random.Random(2)
    primes = pb.pairings_default_moduli(9)
    for m in range(1, 10):
        M = 1
        for p in primes[:m]:
            M *= p
        for _ in range(50):
            x = rng.randrange(-(M // 2) + 1, M // 2)
            assert pb.pairings_crt_signed(primes[:m], [x % p for p in primes[:m]]) == x


def test_reconstruct_against_python_ints(paper_counts):
    primes = pb.pairings_default_moduli(9)
    for (kind, n), S in paper_counts.items():
        if n > 32 or n < 2:
            continue
        m = pb.pairings_min_moduli(kind, n)
        mods = primes[: m + 1]
        H = (2 * S) << (2 * n - 1)
        res = [H % p for p in mods]
        assert pb.pairings_reconstruct(kind, n, mods, res) == (2 * S, S)
        # zero total (n with no pairings)
        assert pb.pairings_reconstruct(kind, n, mods, [0] * len(mods)) == (0, 0)
        # corrupted check prime
        bad = list(res)
        bad[-1] = (bad[-1] + 1) % mods[-1]
        with pytest.raises(pb.PairingsError) as ei:
            pb.pairings_reconstruct(kind, n, mods, bad)
        assert ei.value.code == -7
        # not divisible by 2^(2n-1)
        H2 = H + (1 << (2 * n - 2))
        with pytest.raises(pb.PairingsError) as ei:
            pb.pairings_reconstruct(kind, n, mods, [H2 % p for p in mods])
        assert ei.value.code == -8
        # D odd
        H3 = (2 * S + 1) << (2 * n - 1)
        with pytest.raises(pb.PairingsError) as ei:
            pb.pairings_reconstruct(kind, n, mods, [H3 % p for p in mods])
        assert ei.value.code == -8
        # too few CRT primes for the bound
        if m >= 2:
            short = primes[: m - 1] + [primes[m]]
            with pytest.raises(pb.PairingsError) as ei:
                pb.pairings_reconstruct(kind, n, short, [H % p for p in short])
            assert ei.value.code == -9


def test_journal_roundtrip_and_mismatch(tmp_path):
    path = str(tmp_path / "j.txt")
    moduli = pb.pairings_default_moduli(4)
    assert pb.pairings_journal_load(path, 1, 12, 6, moduli) == ([], [0, 0, 0, 0])
    pb.pairings_journal_append(path, 1, 12, 6, moduli, 0, 8, [1, 2, 3, 4])
    pb.pairings_journal_append(path, 1, 12, 6, moduli, 16, 24, [moduli[0] - 1, 5, 6, 7])
    ranges, total = pb.pairings_journal_load(path, 1, 12, 6, moduli)
    assert ranges == [(0, 8), (16, 24)]
    assert total == [0, 7, 9, 11]
    # torn last line (crash mid-write) is ignored
    with open(path, "ab") as f:
        f.write(b"24 32 1 2")
    ranges, total = pb.pairings_journal_load(path, 1, 12, 6, moduli)
    assert ranges == [(0, 8), (16, 24)]
    # other parameters are refused
    for args in ((0, 12, 6, moduli), (1, 13, 6, moduli), (1, 12, 7, moduli), (1, 12, 6, moduli[:3])):
        with pytest.raises(pb.PairingsError) as ei:
            pb.pairings_journal_load(path, *args)
        assert ei.value.code == -11
    with pytest.raises(pb.PairingsError):
        pb.pairings_journal_append(path, 0, 12, 6, moduli, 32, 40, [0, 0, 0, 0])
    # overlapping ranges would double count
    path2 = str(tmp_path / "j2.txt")
    pb.pairings_journal_append(path2, 1, 12, 6, moduli, 0, 8, [1, 2, 3, 4])
    pb.pairings_journal_append(path2, 1, 12, 6, moduli, 4, 12, [1, 2, 3, 4])
    with pytest.raises(pb.PairingsError):
        pb.pairings_journal_load(path2, 1, 12, 6, moduli)


def test_journal_append_after_a_torn_line_and_strict_lines(tmp_path):
    # a crash in the middle of a write leaves bytes behind the last newline: the next append must cut them off, not
    # glue its own line onto them (the glued line would parse as a valid range with garbage residues)
    path = str(tmp_path / "j.txt")
    moduli = pb.pairings_default_moduli(4)
    pb.pairings_journal_append(path, 1, 12, 6, moduli, 0, 8, [1, 2, 3, 4])
    with open(path, "ab") as f:
        f.write(b"24 32 1 2")
    pb.pairings_journal_append(path, 1, 12, 6, moduli, 32, 40, [100, 200, 300, 400])
    ranges, total = pb.pairings_journal_load(path, 1, 12, 6, moduli)
    assert ranges == [(0, 8), (32, 40)] and total == [101, 202, 303, 404]
    text = open(path).read()
    assert text.endswith("32 40 100 200 300 400\n") and "24 32" not in text
    # a torn HEADER (no complete line at all): the file is started afresh
    path2 = str(tmp_path / "j2.txt")
    with open(path2, "wb") as f:
        f.write(b"pairings-journal v1 kind=1 n=1")
    assert pb.pairings_journal_load(path2, 1, 12, 6, moduli) == ([], [0, 0, 0, 0])
    pb.pairings_journal_append(path2, 1, 12, 6, moduli, 8, 16, [5, 6, 7, 8])
    assert pb.pairings_journal_load(path2, 1, 12, 6, moduli) == ([(8, 16)], [5, 6, 7, 8])
    # lines with surplus, missing or non-numeric tokens, signs, overflowing numbers, residues >= p: refused
    header = open(path).read().splitlines()[0]
    for bad in ("0 8 1 2 3 4 5", "0 8 1 2 3", "0 8 1 2 x 4", "0 -8 1 2 3 4", "+0 8 1 2 3 4", "0 8 1 2 3 99999999999999999999999",
                "0 8 1 2 3 %d" % moduli[3], "8 8 1 2 3 4", "0 65 1 2 3 4", "0x0 8 1 2 3 4", "0 8 1 2 3 4\t5", ""):
        p3 = str(tmp_path / "bad.txt")
        with open(p3, "w") as f:
            f.write(header + "\n" + bad + "\n")
        with pytest.raises(pb.PairingsError) as ei:
            pb.pairings_journal_load(p3, 1, 12, 6, moduli)
        assert ei.value.code == -11, bad
    # many lines: the overlap check is sort-based (2^15 ranges load at once)
    p4 = str(tmp_path / "big.txt")
    with open(p4, "w") as f:
        f.write("pairings-journal v1 kind=0 n=24 chunk_bits=20 moduli=" + ",".join(map(str, moduli)) + "\n")
        for j in range(1 << 15):
            f.write("%d %d 1 1 1 1\n" % (32 * j, 32 * j + 32))
    ranges, total = pb.pairings_journal_load(p4, 0, 24, 20, moduli)
    assert len(ranges) == 1 << 15 and total == [1 << 15] * 4


def test_journal_merge_puts_rank_journals_together(tmp_path):
    # PAPER.md:253 "simply put the result together at the end"; PAPER.md:257 (4 .. 1024 GPU jobs)
    moduli = pb.pairings_default_moduli(4)
    kind, n, C = 1, 12, 6
    rnd = random.Random(5)
    paths, want, rows = [], [0] * 4, {}
    for r in range(3):
        b, e = pb.pairings_rank_range(C, r, 3)
        path = str(tmp_path / ("rank%d.txt" % r))
        for lo in range(b, e, 5):
            hi = min(lo + 5, e)
            row = [rnd.randrange(p) for p in moduli]
            pb.pairings_journal_append(path, kind, n, C, moduli, lo, hi, row)
            want = [(w + v) % p for w, v, p in zip(want, row, moduli)]
        paths.append(path)
    out = str(tmp_path / "merged.txt")
    nr, total, covered = pb.pairings_journal_merge(paths[::-1], kind, n, C, moduli, out)
    assert total == want and covered == 1 << C and nr == 15
    ranges, t2 = pb.pairings_journal_load(out, kind, n, C, moduli)
    assert t2 == want and ranges == sorted(ranges) and ranges[0][0] == 0 and ranges[-1][1] == 1 << C
    # partial coverage is reported, not an error
    nr, total, covered = pb.pairings_journal_merge(paths[:2], kind, n, C, moduli)
    assert covered == pb.pairings_rank_range(C, 1, 3)[1]
    # the same journal twice = every chunk counted twice: refused; so are a foreign journal and a missing file
    for bad in (paths + [paths[0]], paths + [str(tmp_path / "nothing.txt")]):
        with pytest.raises(pb.PairingsError) as ei:
            pb.pairings_journal_merge(bad, kind, n, C, moduli)
        assert ei.value.code == -11
    foreign = str(tmp_path / "foreign.txt")
    pb.pairings_journal_append(foreign, kind, 11, C, moduli, 0, 1, [0, 0, 0, 0])
    with pytest.raises(pb.PairingsError):
        pb.pairings_journal_merge([paths[0], foreign], kind, n, C, moduli)


def test_mode_rule_of_lemma24_lives_behind_the_abi(tmp_path):
    # Lemma 2.4: the x_2 = +1 half is the chunk range [0, 2^(C-1)); equal halves -> factor 2,
    # cancelling halves -> nothing to evaluate, H = 0.  Pairings exist exactly when the halves are equal.
    moduli = pb.pairings_default_moduli(4)
    assert pb.pairings_mode_chunks(1, 12, 6, 0) == (64, 1)
    assert pb.pairings_mode_chunks(1, 12, 6, pb.RUN_LEMMA24) == (32, 2)            # L(12) exists
    assert pb.pairings_mode_chunks(1, 12, 0, pb.RUN_LEMMA24) == (1, 1)             # no chunk bit to fix: flag ignored
    assert pb.pairings_mode_chunks(0, 14, 6, pb.RUN_LEMMA24) == (0, 0)             # S(14) does not exist: halves cancel
    assert pb.pairings_mode_chunks(0, 13, 6, pb.RUN_LEMMA24 | pb.RUN_AUDIT) == (32, 2)
    for kind in (0, 1):
        for n in range(2, 33):
            exists = n % 4 in ((0, 1) if kind == 0 else (0, 3))
            assert pb.pairings_mode_chunks(kind, n, 3, pb.RUN_LEMMA24) == ((4, 2) if exists else (0, 0))
    with pytest.raises(pb.PairingsError):
        pb.pairings_mode_chunks(1, 12, 6, 64)                                      # unknown flag
    raw = [5, moduli[1] - 1, 0, 7]
    assert pb.pairings_finish_total(1, 12, 6, 0, 64, moduli, raw) == (True, raw)
    assert pb.pairings_finish_total(1, 12, 6, 0, 63, moduli, raw) == (False, raw)
    assert pb.pairings_finish_total(1, 12, 6, pb.RUN_LEMMA24, 32, moduli, raw) == (True, [10, moduli[1] - 2, 0, 14])
    assert pb.pairings_finish_total(1, 12, 6, pb.RUN_LEMMA24, 31, moduli, raw) == (False, raw)
    assert pb.pairings_finish_total(0, 14, 6, pb.RUN_LEMMA24, 0, moduli, raw) == (True, [0, 0, 0, 0])
    with pytest.raises(pb.PairingsError) as ei:
        pb.pairings_finish_total(1, 12, 6, pb.RUN_LEMMA24, 33, moduli, raw)        # rows of the other half got in
    assert ei.value.code == -3
    # merging in a mode: ranges outside the evaluated half are refused, whatever their total length
    kind, n, C = 1, 12, 6
    good, mixed, full = (str(tmp_path / f) for f in ("good.txt", "mixed.txt", "full.txt"))
    row = [1, 2, 3, 4]
    pb.pairings_journal_append(good, kind, n, C, moduli, 0, 16, row)
    pb.pairings_journal_append(good, kind, n, C, moduli, 16, 32, row)
    assert pb.pairings_journal_merge_mode([good], kind, n, C, moduli, pb.RUN_LEMMA24) == (2, [2, 4, 6, 8], 32, 32)
    pb.pairings_journal_append(mixed, kind, n, C, moduli, 0, 16, row)              # 16 chunks of each half: length 32
    pb.pairings_journal_append(mixed, kind, n, C, moduli, 32, 48, row)
    assert pb.pairings_journal_merge([mixed], kind, n, C, moduli)[2] == 32   # mode-less merge: plain coverage
    with pytest.raises(pb.PairingsError) as ei:
        pb.pairings_journal_merge_mode([mixed], kind, n, C, moduli, pb.RUN_LEMMA24)
    assert ei.value.code == -11
    pb.pairings_journal_append(full, kind, n, C, moduli, 0, 64, row)               # a job run without the symmetry
    with pytest.raises(pb.PairingsError):
        pb.pairings_journal_merge_mode([full], kind, n, C, moduli, pb.RUN_LEMMA24)
    assert pb.pairings_journal_merge_mode([full], kind, n, C, moduli, 0) == (1, row, 64, 64)


def test_pt_counts_conventions():
    # the conventions differ by exactly a factor of two (n > 1); Table 6 caption prints the identified count
    import math
    d, s_ = pb.pairings_pt_counts(12, math.log(455936.0))
    assert abs(d - 455936.0) < 1e-6 and s_ == d / 2                 # S(12) = 227,968
    with pytest.raises(pb.PairingsError):
        pb.pairings_pt_counts(12, float("inf"))
    with pytest.raises(pb.PairingsError):
        pb.pairings_pt_counts(1, 0.0)


def test_duplicate_run_vote_all_outcomes():
    # every job twice, "if there was a mismatch the job was ran a third time to establish a match"
    a, b, c = [1, 2, 3, 4], [1, 2, 3, 5], [9, 9, 9, 9]
    assert pb.pairings_vote_rows(a, list(a)) == 0
    assert pb.pairings_vote_rows(a, b) == 3                       # third run needed
    assert pb.pairings_vote_rows(a, b, list(a)) == 0              # third confirms the first
    assert pb.pairings_vote_rows(a, b, list(b)) == 1              # third confirms the second
    with pytest.raises(pb.PairingsError) as ei:
        pb.pairings_vote_rows(a, b, c)                            # no two agree
    assert ei.value.code == -7
    # the driver: which attempts are evaluated, which rows win
    for script, want_rows, want_mm, want_calls in (
            ({0: a, 1: list(a)}, a, 0, [0, 1]),
            ({0: a, 1: b, 2: list(a)}, a, 1, [0, 1, 2]),
            ({0: a, 1: b, 2: list(b)}, b, 1, [0, 1, 2])):
        calls = []
        rows, mm = pb.pairings_duplicate_vote(lambda k: (calls.append(k), script[k])[1], 4)
        assert (rows, mm, calls) == (want_rows, want_mm, want_calls)
    with pytest.raises(pb.PairingsError) as ei:
        pb.pairings_duplicate_vote(lambda k: {0: a, 1: b, 2: c}[k], 4)
    assert ei.value.code == -7
    with pytest.raises(pb.PairingsError) as ei:                   # an evaluation error is passed through
        pb.pairings_duplicate_vote(lambda k: -6 if k == 1 else a, 4)
    assert ei.value.code == -6
    # an evaluator that raises must not look like two agreeing all-zero attempts (ctypes swallows callback exceptions)
    def broken(k):
        raise KeyError("attempt %d failed" % k)
    with pytest.raises(KeyError):
        pb.pairings_duplicate_vote(broken, 4)
    with pytest.raises(ValueError):
        pb.pairings_duplicate_vote(lambda k: [1, 2, 3], 4)        # a short row would leave a word unfilled


def test_run_slice_argument_checks_need_no_gpu():
    moduli = pb.pairings_default_moduli(4)
    # a slice of a job whose halves cancel (no pairing exists): nothing to evaluate
    assert pb.pairings_run_slice(pb.SKOLEM, 10, 8, moduli, 64, 32, 96, None, 0, 0, None, pb.RUN_LEMMA24) == ([0] * 4, 0, 0)
    # a slice entirely in the x_2 = -1 half of a symmetric job: nothing to evaluate either
    assert pb.pairings_run_slice(pb.SKOLEM, 12, 8, moduli, 64, 128, 256, None, 0, 0, None, pb.RUN_LEMMA24) == ([0] * 4, 0, 0)
    for b, e in ((5, 4), (0, 257)):
        with pytest.raises(pb.PairingsError) as ei:
            pb.pairings_run_slice(pb.SKOLEM, 12, 8, moduli, 64, b, e)
        assert ei.value.code == -3


def test_compute_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(pb.PairingsError) as ei:
        pb.count_pairings_host(1, 12, 6, 0, 4, pb.pairings_default_moduli(4))
    assert ei.value.code == -6
    with pytest.raises(pb.PairingsError):
        pb.pairings_run(1, 12, 6, pb.pairings_default_moduli(4), 16)


def test_lemma24_applies_exactly_where_pairings_exist():
    # PAPER.md:41,49 (existence) and PAPER.md:215-249 (Lemma 2.4; the Langford case by the same argument)
    for n in range(2, 33):
        assert pb.pairings_lemma24(pb.SKOLEM, n) == (1 if n % 4 in (0, 1) else 0)
        assert pb.pairings_lemma24(pb.LANGFORD, n) == (1 if n % 4 in (0, 3) else 0)
    with pytest.raises(pb.PairingsError):
        pb.pairings_lemma24(pb.SKOLEM, 1)
    with pytest.raises(pb.PairingsError):
        pb.pairings_lemma24(2, 8)


def test_run_ex_without_pairings_needs_no_gpu():
    # term(x^) = -term(x): the two x_2 halves cancel, H = 0, nothing is launched (so this runs on CPU)
    moduli = pb.pairings_default_moduli(4)
    total, done, needed = pb.pairings_run_ex(pb.SKOLEM, 10, 8, moduli, 64, None, 0, 0, None, pb.RUN_LEMMA24)
    assert (total, done, needed) == ([0, 0, 0, 0], 0, 0)
    assert pb.pairings_reconstruct(pb.SKOLEM, 10, moduli, total) == (0, 0)
    with pytest.raises(pb.PairingsError):
        pb.pairings_run_ex(pb.SKOLEM, 10, 8, moduli, 64, None, 0, 0, None, 8)      # unknown flag


def test_pt_draw_counter_must_not_wrap():
    # the draw counter ((r (T+1) + tt) M + j) S + slot must stay below 2^64, else two replicas would share a random stream
    # (the oracle wraps the same way, so parity could not show it): refused before anything is launched
    betas = [0.0] + [0.5 * i for i in range(1, 32)]
    with pytest.raises(pb.PairingsError) as ei:
        pb.pairings_pt_run(pb.SKOLEM, 32, betas, 0, 1 << 30, 1 << 25, 0, 1, 0, 0, 0, 0)       # 2^30 * 2^25 * 32 * 32 = 2^65
    assert ei.value.code == -10
    with pytest.raises(pb.PairingsError) as ei:
        pb.pairings_pt_run(pb.SKOLEM, 12, betas[:12], 0, 1 << 30, 1 << 25, 0, 1, 0, 0, 0, 0)  # in range: next check is the NULL pointers
    assert ei.value.code == -5

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
    for code in range(-11, 0):
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
        pb.pairings_run_ex(pb.SKOLEM, 10, 8, moduli, 64, None, 0, 0, None, 4)      # unknown flag

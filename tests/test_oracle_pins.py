"""Pins for the CPU oracle (oracle/godfrey_oracle.cpp) against what the paper and the mathematics fix.

None of these touches the CUDA path.  Each pin names the passage of /root/reference/PAPER.md it
comes from; together they are chosen so that a dropped term, a wrong sign or index, a wrong
distance convention or a transposed operand in the oracle fails at least one of them.
"""
import itertools
import math
import random

import pytest

import oracle

S, L = oracle.SKOLEM, oracle.LANGFORD
THREADS = 8


def dist(kind, k):
    return k if kind == S else k + 1


def exists(kind, n):
    # PAPER.md:41 (Skolem iff n = 0,1 mod 4), PAPER.md:49 (Langford iff n = 0,3 mod 4)
    return n % 4 in ((0, 1) if kind == S else (0, 3))


def is_valid_sequence(kind, seq):
    n = len(seq) // 2
    for k in range(1, n + 1):
        pos = [i for i, v in enumerate(seq, start=1) if v == k]
        if len(pos) != 2 or pos[1] - pos[0] != dist(kind, k):
            return False
    return True


# ------------------------------------------------------------------ backtracking enumerator pins

def test_brute_lists_the_six_n4_sequences(worked_examples):
    # coefficient 6, and the six sequences printed there
    cnt, seqs = oracle.brute_list(S, 4)
    assert cnt == 6
    assert set(seqs) == set(worked_examples["SKOLEM4"])
    assert len(set(worked_examples["SKOLEM4"])) == 6


def test_brute_contains_paper_example_pairings(worked_examples):
    # PAPER.md:27 Skolem n=4 pairs (7,8)(3,5)(1,4)(2,6)
    pairs = worked_examples["PAIRS_S4"][0]
    seq = [0] * 8
    for k in range(4):
        a, b = pairs[2 * k], pairs[2 * k + 1]
        assert b - a == k + 1
        seq[a - 1] = seq[b - 1] = k + 1
    assert tuple(seq) in set(oracle.brute_list(S, 4)[1])
    # PAPER.md:33 Langford n=4: 2,3,4,2,1,3,1,4 (the two k's are k+1 positions apart)
    lang = worked_examples["LANGFORD4"][0]
    assert is_valid_sequence(L, lang)
    cnt, seqs = oracle.brute_list(L, 4)
    assert cnt == 2 and lang in set(seqs) and tuple(reversed(lang)) in set(seqs)
    # PAPER.md:35-39 Nickerson n=5 == Skolem pairs (8,9)(3,5)(1,4)(6,10)(2,7)
    nick = worked_examples["NICKERSON5"][0]
    pairs = worked_examples["PAIRS_S5"][0]
    seq = [0] * 10
    for k in range(5):
        a, b = pairs[2 * k], pairs[2 * k + 1]
        assert b - a == k + 1
        seq[a - 1] = seq[b - 1] = k + 1
    assert tuple(seq) == nick
    assert nick in set(oracle.brute_list(S, 5)[1])
    # PAPER.md:63 the reflected pair are two distinct Skolem sequences
    a, b = worked_examples["REFLECTED"]
    assert a == tuple(reversed(b)) and a != b
    assert {a, b} <= set(oracle.brute_list(S, 4)[1])


def test_brute_every_listed_sequence_is_valid_and_distinct():
    for kind, n in ((S, 8), (L, 8), (S, 9), (L, 7)):
        cnt, seqs = oracle.brute_list(kind, n, 4096)
        assert cnt == len(seqs) == len(set(seqs))
        assert all(is_valid_sequence(kind, s) for s in seqs)
        # no palindromes, reflections come in pairs
        assert all(tuple(reversed(s)) in set(seqs) and tuple(reversed(s)) != s for s in seqs)


@pytest.mark.parametrize("kind,n", [(S, n) for n in range(2, 14)] + [(L, n) for n in range(2, 13)])
def test_brute_matches_paper_tables(kind, n, paper_counts):
    # Tables 7 and 8, reflections identified; D = 2 x that
    d = oracle.brute_count(kind, n)
    if exists(kind, n):
        assert d == 2 * paper_counts[(kind, n)]
    else:
        assert d == 0


# ------------------------------------------------------------------ formula: single terms

@pytest.mark.parametrize("n", [2, 3, 4, 5, 8, 12, 13, 20, 24, 32])
def test_term_all_plus_closed_form(n):
    # F has (2n-1)!/(n-1)! monomials, so F(n, all +1) is that number (Skolem);
    # Langford: prod_k (2n-k-1) = (2n-2)!/(n-2)!
    x = [1] * (2 * n)
    assert oracle.term(S, n, x) == math.factorial(2 * n - 1) // math.factorial(n - 1)
    assert oracle.term(L, n, x) == math.factorial(2 * n - 2) // math.factorial(n - 2)


@pytest.mark.parametrize("kind", [S, L])
@pytest.mark.parametrize("n", [2, 3, 4, 7, 12, 21, 32])
def test_term_alternating_vector(kind, n):
    # x_i = (-1)^i: every summand of P_k is (-1)^{d_k}, so P_k = (-1)^{d_k} (2n - d_k)
    x = [(-1) ** i for i in range(1, 2 * n + 1)]
    expect = (-1) ** n  # sign = prod_i (-1)^i = (-1)^{n(2n+1)}
    for k in range(1, n + 1):
        d = dist(kind, k)
        expect *= (-1) ** d * (2 * n - d)
    assert oracle.term(kind, n, x) == expect


@pytest.mark.parametrize("kind", [S, L])
def test_term_single_flip_closed_form(kind):
    # all +1 except x_j = -1: P_k = (2n-d_k) - 2*[j-d_k >= 1] - 2*[j+d_k <= 2n], sign = -1.
    # Catches a wrong boundary or a shifted index in the inner sum.
    for n in (4, 9, 16):
        N = 2 * n
        for j in range(1, N + 1):
            x = [1] * N
            x[j - 1] = -1
            expect = -1
            for k in range(1, n + 1):
                d = dist(kind, k)
                expect *= (N - d) - 2 * (j - d >= 1) - 2 * (j + d <= N)
            assert oracle.term(kind, n, x) == expect


def _python_term(kind, n, x):
    """Independent restatement via autocorrelation of the sign vector (big Python ints)."""
    N = 2 * n
    prod = 1
    for k in range(1, n + 1):
        d = dist(kind, k)
        prod *= sum(a * b for a, b in zip(x[: N - d], x[d:]))
    return prod * (-1) ** sum(1 for v in x if v == -1)


@pytest.mark.parametrize("kind", [S, L])
@pytest.mark.parametrize("n", [5, 12, 24, 32])
def test_term_random_vectors_bigint(kind, n):
    # exercises the oracle's own big integer at sizes beyond 64/128 bits
    rng = random.Random(150700315 + 97 * n + kind)
    for _ in range(200):
        x = [rng.choice((1, -1)) for _ in range(2 * n)]
        assert oracle.term(kind, n, x) == _python_term(kind, n, x)


@pytest.mark.parametrize("kind", [S, L])
@pytest.mark.parametrize("n", [4, 5, 7, 8, 12, 13, 19, 20])
def test_symmetry_lemmas(kind, n):
    rng = random.Random(7 * n + kind)
    for _ in range(100):
        x = [rng.choice((1, -1)) for _ in range(2 * n)]
        t = oracle.term(kind, n, x)
        # Lemma 2.2: negation
        assert t == oracle.term(kind, n, [-v for v in x])
        # Lemma 2.3 (reading A10): F(n,X) = F(n, reverse X)
        assert oracle.F(kind, n, x) == oracle.F(kind, n, x[::-1])
        # Lemma 2.4: negate even positions, valid when pairings exist
        xhat = [v if p % 2 == 1 else -v for p, v in enumerate(x, start=1)]
        if exists(kind, n):
            assert t == oracle.term(kind, n, xhat)
        else:
            assert t == -oracle.term(kind, n, xhat)


# ------------------------------------------------------------------ formula: sums

def _expand_coefficient(kind, n):
    """Coefficient of x_1...x_2n in F(n,X) by brute-force expansion."""
    N = 2 * n
    poly = {(0,) * N: 1}
    for k in range(1, n + 1):
        d = dist(kind, k)
        nxt = {}
        for mono, c in poly.items():
            for i in range(N - d):
                if mono[i] or mono[i + d]:
                    continue  # a squared variable can never lead to x_1...x_2n
                m = list(mono)
                m[i] = m[i + d] = 1
                m = tuple(m)
                nxt[m] = nxt.get(m, 0) + c
        poly = nxt
    return poly.get((1,) * N, 0)


@pytest.mark.parametrize("kind,n", [(S, 4), (S, 5), (L, 3), (L, 4), (S, 3), (L, 5)])
def test_sum_equals_coefficient_of_full_monomial(kind, n):
    # Lemma 2.1: Sigma_full = 2^{2n} x coefficient of x_1...x_2n
    s, _ = oracle.total(kind, n)
    assert s == (1 << (2 * n)) * _expand_coefficient(kind, n)


def test_n4_coefficient_is_six():
    # PAPER.md:158
    assert oracle.count_distinct(S, 4) == 6
    assert _expand_coefficient(S, 4) == 6


@pytest.mark.parametrize("kind,n", [(k, n) for k in (S, L) for n in range(2, 12)])
def test_formula_equals_backtracking_small(kind, n):
    d = oracle.count_distinct(kind, n, THREADS)
    assert d == oracle.brute_count(kind, n)
    assert d % 2 == 0
    if not exists(kind, n):
        assert d == 0


@pytest.mark.parametrize("kind,n", [(L, 12), (S, 12), (S, 13)])
def test_formula_equals_backtracking_and_paper_n12_13(kind, n, paper_counts):
    # BASELINE configs 1 and 2: L(12) = 108,144, S(13) = 1,520,280
    d = oracle.count_distinct(kind, n, THREADS)
    assert d == oracle.brute_count(kind, n) == 2 * paper_counts[(kind, n)]


def test_paper_distinct_tables_are_twice_identified(paper_counts, paper_distinct):
    # a consistency check of the fixtures themselves
    for key, v in paper_distinct.items():
        assert v == 2 * paper_counts[key]


def test_negation_symmetry_halves_the_sum():
    # Lemma 2.2: the x_1 = +1 half (index < 2^{2n-1}) is exactly half of Sigma_full
    for kind, n in ((S, 5), (L, 7), (S, 8)):
        full, _ = oracle.total(kind, n, THREADS)
        half, _, _ = oracle.range_sum(kind, n, 0, 1 << (2 * n - 1))
        assert 2 * half == full


@pytest.mark.parametrize("kind,n,C", [(S, 5, 0), (S, 5, 3), (L, 7, 5), (S, 8, 6), (L, 8, 15)])
def test_chunks_partition_the_half_sum(kind, n, C):
    moduli = [2147483647, 2147483629, 2147483587]
    full, nz_full = oracle.total(kind, n, THREADS)
    acc, nz = 0, 0
    for c in range(1 << C):
        t, z, res = oracle.chunk(kind, n, C, c, moduli)
        assert res == [t % p for p in moduli]  # mathematical mod, in [0,p) (reading A8)
        acc += t
        nz += z
    assert 2 * acc == full
    assert 2 * nz == nz_full


def test_chunk_index_contract():
    # bit b of v <-> position 2n-b; chunk c fixes x_2..x_{C+1}, msb of c <-> x_2.
    kind, n, C = S, 4, 3
    N = 2 * n
    for c in range(1 << C):
        want = 0
        for low in itertools.product((1, -1), repeat=N - 1 - C):
            pre = [1] + [(-1 if (c >> (C - 1 - i)) & 1 else 1) for i in range(C)]
            want += oracle.term(kind, n, pre + list(low))
        assert oracle.chunk(kind, n, C, c)[0] == want


@pytest.mark.parametrize("kind,n", [(k, n) for k in (S, L) for n in range(2, 10)])
def test_lemma24_x2_half_is_half_the_sum_or_cancels(kind, n):
    # Lemma 2.4 as the host driver uses it: chunk bit C-1 is x_2, so with C = 1 chunk 0
    # is the x_2 = +1 half.  Where pairings exist both halves are equal; elsewhere they cancel.
    t0, t1 = oracle.chunk(kind, n, 1, 0)[0], oracle.chunk(kind, n, 1, 1)[0]
    exists = (n % 4 in (0, 1)) if kind == S else (n % 4 in (0, 3))
    if exists:
        assert t0 == t1 and 2 * t0 == oracle.brute_count(kind, n) << (2 * n - 1)
    else:
        assert t0 == -t1 and oracle.brute_count(kind, n) == 0


@pytest.mark.parametrize("kind,n", [(S, 4), (S, 5), (S, 8), (L, 7), (L, 8), (S, 13), (L, 20), (S, 21), (S, 24)])
def test_sign_of_a_term_is_the_parity_of_the_distance_n_sum(kind, n):
    # The pairs (i, i+n), i = 1..n, cover every position exactly once, so #(x_i != x_{i+n}) = (n - P_n)/2 has the
    # parity of #(x_i = -1) and prod_i x_i = (-1)^{(n - P_n)/2}.  (The SWAR kernel does not store the sign of a
    # queued term, it reads it off the distance-n sum; both kinds have a pair of distance n.)
    rng = random.Random(1000 * kind + n)
    assert n in [(k if kind == S else k + 1) for k in range(1, n + 1)]
    for _ in range(200):
        x = [rng.choice((1, -1)) for _ in range(2 * n)]
        Pn = sum(x[i] * x[i + n] for i in range(n))
        assert (n - Pn) % 2 == 0
        assert math.prod(x) == (-1) ** ((n - Pn) // 2)

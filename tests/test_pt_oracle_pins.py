"""Pins of the approximate-counting oracle (oracle/pt_oracle.cpp; §3, Algorithm 2) against things
other than itself: exhaustive enumeration, closed forms, the paper's printed counts and its Table 6."""
import math
import os
import statistics

import pytest

from oracle import pt

S, L = 0, 1
GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def table6():
    rows = []
    for ln in open(os.path.join(GOLD, "paper_table6.txt")):
        if ln.strip() and not ln.startswith("#"):
            f = ln.split()
            rows.append(dict(i=int(f[0]), beta=float(f[1]), W1=float(f[2]), W2=float(f[3]), E=float(f[4]), ratio=float(f[5])))
    return rows


def test_generator_is_splitmix64():
    # draw(seed, ctr) = output ctr+1 of SplitMix64 started at `seed`; the first outputs for seed 0 are the
    # widely published ones, and the mixing function restated here in Python gives the rest
    def mix(z):
        z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9 & (2**64 - 1)
        z = (z ^ (z >> 27)) * 0x94D049BB133111EB & (2**64 - 1)
        return z ^ (z >> 31)
    assert pt.draw(0, 0) == 0xE220A8397B1DCDAF
    assert pt.draw(0, 1) == 0x6E789E6AA1B965F4
    for seed, ctr in ((1, 0), (150700315, 12345), (2**64 - 1, 2**40)):
        assert pt.draw(seed, ctr) == mix((seed + 0x9E3779B97F4A7C15 * (ctr + 1)) & (2**64 - 1))


@pytest.mark.parametrize("kind,n,pairings", [(S, 4, 6), (S, 5, 10), (S, 6, 0), (S, 7, 0), (L, 3, 2), (L, 4, 2),
                                             (L, 5, 0), (L, 7, 52)])
def test_density_of_states_closed_forms(kind, n, pairings):
    g = pt.density_of_states(kind, n)
    d = [k if kind == S else k + 1 for k in range(1, n + 1)]
    assert sum(g) == math.prod(2 * n - dk for dk in d)              # Z(0)
    if kind == S:
        assert sum(g) == math.factorial(2 * n - 1) // math.factorial(n - 1)
    assert g[0] == pairings                                           # PAPER.md:158 (6), Tables 7/8 doubled (:63)
    assert g[2 * n] == 0 and g[2 * n - 1] == 0                        # at least two bins are occupied


def runs(kind, n, betas, replicas, iterations, seeds):
    out = []
    for s in seeds:
        hist, mv, sw = pt.run(kind, n, betas, replicas, iterations, s)
        out.append((hist, mv, sw, pt.ratios(kind, n, betas, hist)))
    return out


@pytest.mark.parametrize("kind,n,betas", [(S, 5, [0, 0.7, 1.5, 2.5, 4.0, 8.0]), (L, 4, [0, 1.0, 2.2, 4.0]),
                                          (S, 4, [0, 0.9, 2.0, 3.5, 7.0])])
def test_monte_carlo_ratios_match_exact_partition_function(kind, n, betas):
    g = pt.density_of_states(kind, n)
    seeds = list(range(101, 113))
    # Algorithm 2 has no burn-in: the first samples of a run come from random configurations, which biases a
    # run of T iterations by O(relaxation time / T); few long replicas and an explicit allowance for it
    reps, T = 1, 1 << 16
    res = runs(kind, n, betas, reps, T, seeds)
    transient = 400.0 / T
    M = len(betas)
    for j in range(M):
        exact = pt.exact_ratio(g, betas[j], betas[j + 1] if j + 1 < M else math.inf)
        vals = [r[3][0][j] for r in res]
        mean, se = statistics.mean(vals), statistics.stdev(vals) / math.sqrt(len(vals))
        assert abs(mean - exact) < 5 * se + transient * exact, (j, mean, exact, se)
    # the final estimate
    est = [math.exp(r[3][1]) for r in res]
    mean, se = statistics.mean(est), statistics.stdev(est) / math.sqrt(len(est))
    assert abs(mean - g[0]) < 5 * se + 0.01 * g[0], (mean, g[0], se)
    # level 1 (beta = 0): every move is accepted and the energy histogram is g(E)/Z(0)
    total = reps * T
    for hist, mv, sw, _ in res:
        assert mv[0] == total and sum(hist[0]) == total and sw[M - 1] == 0
    Z0 = sum(g)
    for E in range(len(g)):
        if g[E] * total / Z0 < 200:
            continue
        freq = [r[0][0][E] / total for r in res]
        mean, se = statistics.mean(freq), statistics.stdev(freq) / math.sqrt(len(freq))
        assert abs(mean - g[E] / Z0) < 5 * se, (E, mean, g[E] / Z0, se)


def test_paper_table6_sample_run_for_s12():
    # the paper's ladder; its estimate 227009 is 0.4 % below the exact 227,968.
    rows = table6()
    betas = [r["beta"] for r in rows]
    replicas, iterations, burn = 4, 1 << 18, 1 << 14                  # ~2^20 counted iterations in total (paper: 2^24)
    hist, mv, sw = pt.run(S, 12, betas, replicas, iterations, 150700315, burn)
    ratios, logz = pt.ratios(S, 12, betas, hist)
    est_identified = math.exp(logz) / 2
    assert abs(est_identified - 227968) < 0.04 * 227968, est_identified
    total = replicas * (iterations - burn)
    for j, r in enumerate(rows):
        w1, w2 = mv[j] / total, sw[j] / total
        mean_e = sum(E * c for E, c in enumerate(hist[j])) / total
        assert abs(w1 - r["W1"]) < 0.03, (j, w1, r["W1"])              # acceptance of new configurations
        if j + 1 < len(rows):
            assert abs(w2 - r["W2"]) < 0.06, (j, w2, r["W2"])          # exchange rate with the next level
        assert abs(mean_e - r["E"]) < 0.15, (j, mean_e, r["E"])        # mean energy
        assert abs(ratios[j] - r["ratio"]) < 0.12 * r["ratio"] + 1e-4, (j, ratios[j], r["ratio"])

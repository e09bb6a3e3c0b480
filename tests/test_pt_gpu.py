"""GPU parity of the approximate counter (pairings_pt_run, §3 Algorithm 2) against the CPU oracle:
the integer counters (energy histograms, accepted moves and exchanges) must be identical, because both sides
draw from the same counter-based generator and take every decision on 32-bit integers."""
import math
import os

import pytest

import paper_1507_00315_b200 as pb
from oracle import pt

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

S, L = pb.SKOLEM, pb.LANGFORD
GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def gpu_counters(kind, n, betas, r0, r1, iterations, burn, seed):
    M, N = len(betas), 2 * n
    hist = torch.zeros((M, N + 1), dtype=torch.int64, device="cuda")
    mv = torch.zeros(M, dtype=torch.int64, device="cuda")
    sw = torch.zeros(M, dtype=torch.int64, device="cuda")
    pb.pairings_pt_run(kind, n, betas, r0, r1, iterations, burn, seed, hist.data_ptr(), mv.data_ptr(), sw.data_ptr(),
                       torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return hist.cpu().tolist(), mv.cpu().tolist(), sw.cpu().tolist()


@pytest.mark.parametrize("kind,n,betas,replicas,iterations,burn,seed", [
    (S, 5, [0, 0.7, 1.5, 2.5, 4.0, 8.0], 64, 512, 0, 1),
    (L, 4, [0, 1.0, 2.2, 4.0], 100, 300, 17, 2),                       # ragged: not a multiple of the block size
    (S, 12, [0, 0.54, 1.1, 1.69, 2.33, 3, 3.73, 4.65, 5.82, 8.1, 16, 32], 70, 400, 100, 150700315),
    (L, 16, [0, 0.5, 1.0, 1.6, 2.3, 3.1, 4.0, 5.2, 7.0, 11.0, 20.0], 33, 200, 0, 7),
    (S, 2, [0], 3, 50, 0, 9),                                          # degenerate: one level, smallest n
    (L, 32, [0, 1.0, 3.0, 9.0], 5, 60, 10, 11),                        # maximum n
])
def test_counters_are_bit_identical_to_the_oracle(kind, n, betas, replicas, iterations, burn, seed):
    want = pt.run(kind, n, betas, replicas, iterations, seed, burn)
    got = gpu_counters(kind, n, betas, 0, replicas, iterations, burn, seed)
    assert got[0] == want[0]
    assert got[1] == want[1] and got[2] == want[2]
    # the library's host-side estimate against the oracle's
    r1, l1 = pb.pairings_pt_estimate(kind, n, betas, got[0]) if all(sum(h) for h in got[0]) and got[0][-1][0] else (None, None)
    if r1 is not None:
        r2, l2 = pt.ratios(kind, n, betas, want[0])
        assert all(abs(a - b) <= 1e-12 * abs(b) for a, b in zip(r1, r2)) and abs(l1 - l2) < 1e-9


def test_replica_ranges_add_up_and_empty_range():
    kind, n, betas = S, 8, [0, 0.8, 1.8, 3.0, 6.0]
    whole = gpu_counters(kind, n, betas, 0, 150, 128, 8, 5)
    a = gpu_counters(kind, n, betas, 0, 37, 128, 8, 5)
    b = gpu_counters(kind, n, betas, 37, 150, 128, 8, 5)
    assert [[x + y for x, y in zip(r, s)] for r, s in zip(a[0], b[0])] == whole[0]
    assert [x + y for x, y in zip(a[1], b[1])] == whole[1] and [x + y for x, y in zip(a[2], b[2])] == whole[2]
    e = gpu_counters(kind, n, betas, 9, 9, 128, 8, 5)
    assert sum(map(sum, e[0])) == 0
    for bad in ([0.5, 1.0], [0, 1.0, 1.0], [0, 2.0, 1.0]):
        with pytest.raises(pb.PairingsError):
            gpu_counters(kind, n, bad, 0, 1, 10, 0, 1)
    with pytest.raises(pb.PairingsError):
        gpu_counters(kind, n, betas, 0, 1, 10, 10, 1)                   # burn_in must be < iterations


def test_table6_ladder_estimates_s12_within_one_percent():
    # PAPER.md:327-342 (ladder), :350 (S(12) = 227,968), "the error found is less than one percent" (:325)
    betas = [float(ln.split()[1]) for ln in open(os.path.join(GOLD, "paper_table6.txt")) if ln.strip() and not ln.startswith("#")]
    # the cold levels need ~10^4 iterations to relax from a random start (no burn-in, 2^13 iterations: -45 %)
    replicas, iterations, burn = 1 << 12, 1 << 15, 1 << 14            # 2^26 counted iterations (paper: 2^24)
    hist, mv, sw = gpu_counters(S, 12, betas, 0, replicas, iterations, burn, 150700315)
    total = replicas * (iterations - burn)
    assert all(sum(h) == total for h in hist) and mv[0] == total
    ratios, logz = pb.pairings_pt_estimate(S, 12, betas, hist)
    est = pb.pairings_pt_counts(12, logz)[1]
    assert est == math.exp(logz) / 2
    assert abs(est - 227968) < 0.01 * 227968, est


@pytest.mark.parametrize("kind,n,exact", [(S, 12, 227968), (S, 16, 700078384), (L, 12, 108144)])
def test_ladder_gives_half_exchange_rates_and_a_good_estimate(kind, n, exact):
    # exchange acceptance "no smaller than one half"; Tables 7/8: approximate within ~1 % of the exact count
    betas = pb.pairings_pt_ladder(kind, n, 0.55, 256, 1 << 14, 7)
    assert betas[0] == 0.0 and all(b > a for a, b in zip(betas, betas[1:])) and 6 <= len(betas) <= 20
    assert betas == pb.pairings_pt_ladder(kind, n, 0.55, 256, 1 << 14, 7)            # deterministic
    r = pb.approx_count(kind, n, 1 << 12, 1 << 16, betas=betas)
    rates = [s / r["samples"] for s in r["swaps"][:-1]]
    assert all(x >= 0.5 for x in rates), rates
    assert abs(r["identified"] - exact) < 0.025 * exact, r["identified"]
    with pytest.raises(pb.PairingsError):
        pb.pairings_pt_ladder(kind, n, 0.55, 256, 1 << 14, 7, cap_levels=3)          # cap reached first

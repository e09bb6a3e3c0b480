"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same chunks; totals against backtracking / the paper's printed values.  Integer work: bit-exact,
zero tolerance."""
import ctypes
import threading

import pytest

import oracle
import paper_1507_00315_b200 as pb
from paper_1507_00315_b200 import seeds

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

S, L = pb.SKOLEM, pb.LANGFORD
VARIANTS = [pb.VARIANT_GENERIC, pb.VARIANT_SWAR]


def gpu_rows(kind, n, C, begin, end, moduli, opts=None, count_nonzero=False):
    m = len(moduli)
    out = torch.full((max(end - begin, 1), m), -1, dtype=torch.int32, device="cuda")
    nz = torch.zeros(1, dtype=torch.int64, device="cuda")
    if opts is None:
        opts = pb.LaunchOpts()
    if count_nonzero:
        opts.nonzero_terms = nz.data_ptr()
    stream = torch.cuda.current_stream().cuda_stream
    pb.count_pairings_ex(kind, n, C, begin, end, moduli, out.data_ptr(), stream, opts)
    torch.cuda.synchronize()
    rows = (out.cpu().to(torch.int64) & 0xFFFFFFFF).tolist()[: end - begin]
    return (rows, int(nz.item())) if count_nonzero else rows


def oracle_rows(kind, n, C, chunks, moduli, threads=8, pieces=1):
    """oracle.chunk for every chunk, on host threads; `pieces` > 1 cuts each chunk's index range into
    equal sub-ranges (oracle.range_sum) whose exact sums are added here, so that a few large chunks
    still use every core."""
    w = 1 << (2 * n - 1 - C)
    jobs = [(i, c * w + j * (w // pieces), c * w + (j + 1) * (w // pieces)) for i, c in enumerate(chunks) for j in range(pieces)]
    parts = [None] * len(jobs)

    def work(tid):
        for k in range(tid, len(jobs), threads):
            parts[k] = oracle.range_sum(kind, n, jobs[k][1], jobs[k][2], moduli)

    ts = [threading.Thread(target=work, args=(t,)) for t in range(threads)]
    [t.start() for t in ts]
    [t.join() for t in ts]
    out = []
    for i in range(len(chunks)):
        mine = [parts[k] for k in range(len(jobs)) if jobs[k][0] == i]
        out.append((sum(p[0] for p in mine), sum(p[1] for p in mine),
                    [sum(p[2][j] for p in mine) % moduli[j] for j in range(len(moduli))]))
    return out


def variant_available(variant, kind, n, C):
    if variant == pb.VARIANT_SWAR:
        return pb.pairings_has_swar(kind, n) and (2 * n - 1 - C) >= 10   # >= 32 prefixes of >= 2^5 steps per chunk
    return True


# ------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("kind,n,C", [(L, 12, 0), (L, 12, 6), (L, 12, 10), (S, 13, 8), (S, 12, 7), (L, 11, 5)])
def test_every_chunk_matches_oracle(kind, n, C, variant):
    if not variant_available(variant, kind, n, C):
        pytest.skip("variant not compiled for this (kind, n)")
    moduli = pb.pairings_default_moduli(4)
    rows, nz = gpu_rows(kind, n, C, 0, 1 << C, moduli, pb.LaunchOpts(variant=variant), count_nonzero=True)
    want = oracle_rows(kind, n, C, list(range(1 << C)), moduli)
    for c in range(1 << C):
        assert rows[c] == want[c][2], (c, rows[c], want[c][2])
        # symmetric CRT lift of the row equals the oracle's exact signed T(c) (reading A8)
        assert pb.pairings_crt_signed(moduli, rows[c]) == want[c][0]
    assert nz == sum(w[1] for w in want)           # early-out statistic phi
    total = pb.pairings_sum_rows(rows, moduli)
    D, Sid = pb.pairings_reconstruct(kind, n, moduli, total)
    assert D == oracle.brute_count(kind, n) and Sid * 2 == D


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("kind,n", [(k, n) for k in (S, L) for n in range(2, 12)])
def test_small_n_totals_match_backtracking(kind, n, variant, paper_counts):
    C = max(0, min(5, 2 * n - 1 - 4))
    if not variant_available(variant, kind, n, C):
        pytest.skip("variant not compiled for this (kind, n)")
    moduli = pb.pairings_default_moduli(pb.pairings_min_moduli(kind, n) + 1)
    rows = gpu_rows(kind, n, C, 0, 1 << C, moduli, pb.LaunchOpts(variant=variant))
    D, Sid = pb.pairings_reconstruct(kind, n, moduli, pb.pairings_sum_rows(rows, moduli))
    assert D == oracle.brute_count(kind, n)
    if (kind, n) in paper_counts:
        assert Sid == paper_counts[(kind, n)]
    else:
        assert D == 0                                # no pairing exists


@pytest.mark.parametrize("variant", VARIANTS)
def test_geometry_never_changes_the_rows(variant):
    kind, n, C = L, 12, 6
    if not variant_available(variant, kind, n, C):
        pytest.skip("variant not compiled")
    moduli = pb.pairings_default_moduli(4)
    ref = gpu_rows(kind, n, C, 0, 1 << C, moduli, pb.LaunchOpts(variant=variant))
    gs = [5, 7, 10] if variant == pb.VARIANT_SWAR else [0, 1, 5, 12, 17]
    for g in gs:
        for threads, bpc in ((32, 1), (128, 2), (256, 1), (64, 8)):
            if bpc * threads > (1 << (2 * n - 1 - C - g)) and (bpc > 1 or variant == pb.VARIANT_SWAR):
                continue
            o = pb.LaunchOpts(variant=variant, gray_bits=g, block_threads=threads, blocks_per_chunk=bpc)
            assert gpu_rows(kind, n, C, 0, 1 << C, moduli, o) == ref, (g, threads, bpc)
    # cutting [0, 2^C) into several calls gives the same rows
    parts = gpu_rows(kind, n, C, 0, 5, moduli) + gpu_rows(kind, n, C, 5, 5, moduli) + \
        gpu_rows(kind, n, C, 5, 64, moduli)
    assert parts == ref
    # another prime set reconstructs the same integers
    other = pb.pairings_default_moduli(9)[5:9]
    rows2 = gpu_rows(kind, n, C, 0, 1 << C, other, pb.LaunchOpts(variant=variant))
    for c in range(1 << C):
        assert pb.pairings_crt_signed(other, rows2[c]) == pb.pairings_crt_signed(moduli, ref[c])


@pytest.mark.parametrize("variant", VARIANTS)
def test_total_independent_of_chunk_bits(variant):
    kind, n = S, 12
    moduli = pb.pairings_default_moduli(4)
    totals = set()
    for C in (0, 3, 9, 14, 19):
        if not variant_available(variant, kind, n, C):
            continue
        rows = gpu_rows(kind, n, C, 0, 1 << C, moduli, pb.LaunchOpts(variant=variant))
        totals.add(tuple(pb.pairings_sum_rows(rows, moduli)))
    assert len(totals) == 1
    assert pb.pairings_reconstruct(kind, n, moduli, list(totals.pop())) == (455936, 227968)


def test_degenerate_geometries_generic():
    # one term per chunk (C = B), n = 2, single modulus, 16 moduli
    for kind, n in ((S, 2), (L, 2), (S, 4), (L, 3)):
        B = 2 * n - 1
        moduli = pb.pairings_default_moduli(2)
        rows = gpu_rows(kind, n, B, 0, 1 << B, moduli, pb.LaunchOpts(variant=pb.VARIANT_GENERIC))
        for c in range(1 << B):
            assert rows[c] == oracle.chunk(kind, n, B, c, moduli)[2]
    m16 = pb.pairings_default_moduli(16)
    rows = gpu_rows(S, 8, 5, 0, 32, m16)
    for c in (0, 7, 31):
        assert rows[c] == oracle.chunk(S, 8, 5, c, m16)[2]
    rows = gpu_rows(S, 8, 5, 3, 9, m16[:1])
    for i, c in enumerate(range(3, 9)):
        assert rows[i] == oracle.chunk(S, 8, 5, c, m16[:1])[2]


def test_maximum_n_32_single_terms():
    # n = 32: N = 64 positions, 63 index bits.  C = B makes every chunk a single sign vector, so the
    # oracle evaluates them one by one (products up to ~2^177: exercises the full product chain).
    moduli = pb.pairings_default_moduli(8)
    for kind in (S, L):
        n, B = 32, 63
        for begin in (0, (1 << 63) - 64, 0x5DEECE66D << 20):
            rows = gpu_rows(kind, n, B, begin, begin + 64, moduli, pb.LaunchOpts(variant=pb.VARIANT_GENERIC))
            for i in range(0, 64, 7):
                assert rows[i] == oracle.chunk(kind, n, B, begin + i, moduli)[2]


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("kind", [S, L])
def test_config3_n16_sampled_chunks_and_total(kind, variant, paper_counts):
    # BASELINE config 3: 2^31 sign vectors, 5 primes + 1 check prime.
    n, moduli = 16, pb.pairings_default_moduli(6)
    if not variant_available(variant, kind, n, 16):
        pytest.skip("variant not compiled")
    C = 16
    chunks = seeds.sample_chunks(C, 16, salt=kind)
    want = oracle_rows(kind, n, C, chunks, moduli)            # 16 x 2^15 terms
    for c, w in zip(chunks, want):
        assert gpu_rows(kind, n, C, c, c + 1, moduli, pb.LaunchOpts(variant=variant))[0] == w[2], c
    if variant == pb.VARIANT_GENERIC and kind == L:
        # the stated geometry: 10 high bits as thread prefix, 21 Gray-code bits per thread (D3)
        rows = gpu_rows(kind, n, 0, 0, 1, moduli, pb.LaunchOpts(variant=variant, gray_bits=21, block_threads=32, blocks_per_chunk=32))
    else:
        rows = gpu_rows(kind, n, 10, 0, 1 << 10, moduli, pb.LaunchOpts(variant=variant))
    D, Sid = pb.pairings_reconstruct(kind, n, moduli, pb.pairings_sum_rows(rows, moduli))
    assert Sid == paper_counts[(kind, n)] and D == 2 * Sid    # 700,078,384 / 326,721,800


def test_host_buffer_call_and_run_driver_with_journal(tmp_path):
    kind, n, C = L, 12, 8
    moduli = pb.pairings_default_moduli(4)
    rows = pb.count_pairings_host(kind, n, C, 10, 20, moduli)
    assert rows == gpu_rows(kind, n, C, 10, 20, moduli)
    path = str(tmp_path / "journal.txt")
    total, done = pb.pairings_run(kind, n, C, moduli, 48, path, max_calls=2)       # interrupted run
    assert done == 96
    ranges, jt = pb.pairings_journal_load(path, kind, n, C, moduli)
    assert ranges == [(0, 48), (48, 96)] and jt == total
    total, done = pb.pairings_run(kind, n, C, moduli, 100, path)                  # resumed
    assert done == 256
    assert pb.pairings_reconstruct(kind, n, moduli, total) == (216288, 108144)
    total2, done2 = pb.pairings_run(kind, n, C, moduli, 256, path)                # nothing left to do
    assert (total2, done2) == (total, 256)
    assert pb.count(S, 13) == (3040560, 1520280)                                 # config 2, both conventions


@pytest.mark.parametrize("kind,n", [(S, 12), (S, 13), (L, 11), (L, 12), (S, 10), (L, 9), (S, 16), (L, 16)])
def test_lemma24_half_run_gives_the_same_count(kind, n, paper_counts, tmp_path):
    # §8(f) NEXT #1: symmetry 3 (Lemma 2.4) in the host driver: half the chunks, doubled
    C = 8
    moduli = pb.pairings_default_moduli(pb.pairings_bound_moduli(kind, n) + 1)
    path = str(tmp_path / "j.txt")
    total, done, needed = pb.pairings_run_ex(kind, n, C, moduli, 48, path, 0, 0, None, pb.RUN_LEMMA24)
    if (kind, n) in paper_counts:
        assert done == needed == 128
        full, fdone = pb.pairings_run(kind, n, C, moduli, 256) if n <= 13 else (total, 256)
        assert total == full and fdone == 256
        D, Sid = pb.pairings_reconstruct(kind, n, moduli, total)
        assert Sid == paper_counts[(kind, n)] and D == 2 * Sid
        # resumed from the complete journal: nothing to do, same answer; a full run refuses nothing either
        assert pb.pairings_run_ex(kind, n, C, moduli, 48, path, 0, 0, None, pb.RUN_LEMMA24) == (total, 128, 128)
    else:
        assert (done, needed) == (0, 0) and pb.pairings_reconstruct(kind, n, moduli, total) == (0, 0)
        full, fdone = pb.pairings_run(kind, n, C, moduli, 256)
        assert pb.pairings_reconstruct(kind, n, moduli, full) == (0, 0)


def test_lemma24_refuses_a_journal_of_the_other_half(tmp_path):
    kind, n, C = L, 12, 6
    moduli = pb.pairings_default_moduli(4)
    path = str(tmp_path / "j.txt")
    pb.pairings_run(kind, n, C, moduli, 64, path)                       # full run: journal covers [0, 64)
    with pytest.raises(pb.PairingsError) as e:
        pb.pairings_run_ex(kind, n, C, moduli, 64, path, 0, 0, None, pb.RUN_LEMMA24)
    assert e.value.code == -11


# ---- BASELINE configs 4 and 5 at full size: rows of seeded chunks against the oracle one by one (each oracle
# chunk is 2^23 .. 2^27 plain evaluations), in the launch geometry bench.py times.  The geometry depends on the
# number of chunks of a launch, so the test asks pairings_query_geometry for the geometry of the bench's launch
# (bench.WL: all 2^16 chunks of L(20) in one call; bench.OTHER_CONFIGS: all 2^18 chunks of S(21); bench.WL24: runs of
# 1024 chunks of S(24)) and pins it on the small launches around the sampled chunks.
def bench_launch_chunks(kind, n, C):
    import bench
    if (kind, n, C) == (bench.WL["kind"], bench.WL["n"], bench.WL["chunk_bits"]):
        return 1 << C
    if (kind, n, C) == (bench.WL24["kind"], bench.WL24["n"], bench.WL24["chunk_bits"]):
        return bench.WL24["run_len"]
    assert any((k, nn, cc) == (kind, n, C) for (k, nn, cc, _m, _r, _w) in bench.OTHER_CONFIGS)
    return 1 << C


@pytest.mark.parametrize("kind,n,C,m,count", [(L, 20, 16, 7, 16), (S, 21, 18, 7, 16), (S, 24, 20, 9, 4)])
def test_full_size_sampled_chunks_match_oracle(kind, n, C, m, count):
    moduli = pb.pairings_default_moduli(m)
    chunks = seeds.sample_chunks(C, count, salt=100 + n)
    want = oracle_rows(kind, n, C, chunks, moduli, threads=16, pieces=16 if n == 24 else 1)
    v, g, t, bpc = pb.pairings_query_geometry(kind, n, C, bench_launch_chunks(kind, n, C))
    assert v == pb.VARIANT_SWAR
    pinned = pb.LaunchOpts(variant=v, gray_bits=g, block_threads=t, blocks_per_chunk=bpc)
    assert pb.pairings_query_geometry(kind, n, C, 8, pinned) == (v, g, t, bpc)       # the pin holds on a small launch
    for i, (c, w) in enumerate(zip(chunks, want)):
        b = min(c & ~7, (1 << C) - 8)
        rows = gpu_rows(kind, n, C, b, b + 8, moduli, pb.LaunchOpts(variant=v, gray_bits=g, block_threads=t, blocks_per_chunk=bpc))
        assert rows[c - b] == w[2], (kind, n, c, "bench geometry", g, t, bpc)
        assert pb.pairings_crt_signed(moduli, rows[c - b]) == w[0]
        # the library's own choice for a 64-chunk launch (several blocks per chunk, atomic mod-add of the block sums)
        b = min(c & ~63, (1 << C) - 64)
        rows = gpu_rows(kind, n, C, b, b + 64, moduli)
        assert rows[c - b] == w[2], (kind, n, c, "default geometry")
        if i < 4:
            # every other Gray-bit count the outer-flip dispatch of this instance has (per-row, not through a sum)
            for g2 in range(max(g - 3, 5), min(n - 2, 16) + 1):
                for bpc2 in (1, 4):
                    if 2 * n - 1 - C - g2 < (t * bpc2).bit_length() - 1:
                        continue                                       # fewer prefixes than threads
                    o = pb.LaunchOpts(variant=v, gray_bits=g2, block_threads=t, blocks_per_chunk=bpc2)
                    assert gpu_rows(kind, n, C, c, c + 1, moduli, o)[0] == w[2], (kind, n, c, g2, bpc2)


@pytest.mark.parametrize("kind,n,C", [(L, 20, 16), (S, 20, 16), (S, 21, 18)])
def test_full_totals_match_the_paper(kind, n, C, paper_counts):
    # PAPER.md:353-354 (Table 7: S(20), S(21)), :380 (Table 8: L(20)); one launch over every chunk, as in bench.py
    moduli = pb.pairings_default_moduli(7)
    out = torch.empty((1 << C, 7), dtype=torch.int32, device="cuda")
    pb.count_pairings(kind, n, C, 0, 1 << C, moduli, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    flat = (ctypes.c_uint32 * ((1 << C) * 7)).from_buffer_copy(out.cpu().numpy().tobytes())
    D, Sid = pb.pairings_reconstruct(kind, n, moduli, pb.pairings_sum_rows(flat, moduli))
    assert Sid == paper_counts[(kind, n)] and D == 2 * Sid
    # and with symmetry 3: half the work
    assert pb.count(kind, n, lemma24=True) == (D, Sid)


@pytest.mark.parametrize("kind,n", [(S, 24), (L, 24)])
def test_full_n24_counts_match_the_paper(kind, n, paper_counts, paper_distinct):
    # BASELINE.json configs[4]: "full run matched against the paper's printed S(24) if within budget" — it is: 2^46 sign
    # vectors (symmetry 3: the x_2 = +1 half of the 2^47) in about 70 s.  S(24) = 102,388,058,845,620,672 (PAPER.md:9,
    # Table 4 :103), A004075(24) = 204,776,117,691,241,344 (:109); L(24) = 46,845,158,056,515,936 (Table 8, :382).
    D, Sid = pb.count(kind, n, lemma24=True)
    assert Sid == paper_counts[(kind, n)] and D == 2 * Sid
    assert Sid == (102388058845620672 if kind == S else 46845158056515936)
    if (kind, n) in paper_distinct:
        assert D == paper_distinct[(kind, n)]


@pytest.mark.parametrize("kind,n,C", [(L, 12, 6), (S, 13, 8), (L, 8, 3), (S, 16, 10)])
def test_duplicate_run_mode_and_tight_moduli(kind, n, C, paper_counts):
    # §8(f) NEXT #3 (every job twice, third run on mismatch) and NEXT #2 (tight prime budget)
    moduli = pb.pairings_default_moduli(pb.pairings_min_moduli(kind, n) + 1)
    assert len(moduli) <= pb.pairings_bound_moduli(kind, n) + 1
    total, done, needed = pb.pairings_run_ex(kind, n, C, moduli, 1 << max(C - 2, 0), None, 0, 0, None,
                                             pb.RUN_DUPLICATE | pb.RUN_LEMMA24)
    assert done == needed == 1 << (C - 1) and pb.pairings_run_ex.last_mismatches == 0
    D, Sid = pb.pairings_reconstruct(kind, n, moduli, total)
    assert Sid == paper_counts[(kind, n)] and D == 2 * Sid
    assert pb.count(kind, n, duplicate=True, tight_moduli=True) == (D, Sid)


# ---- the remaining exact values of Tables 7/8 the SWAR kernel is compiled for
# (L(7) at C = 3 is the only geometry that launches swar_kernel<1,7>; S(8), L(8), S(20) were checked through totals only,
# L(24) not at all before round 3)
@pytest.mark.parametrize("kind,n,C,count,pieces", [(L, 7, 3, 8, 1), (L, 7, 0, 1, 1), (S, 8, 4, 16, 1), (L, 8, 4, 16, 1),
                                                   (S, 20, 16, 8, 1), (L, 24, 20, 3, 16),
                                                   (S, 9, 4, 16, 1), (L, 15, 12, 8, 1), (S, 17, 16, 8, 1), (L, 19, 20, 8, 1),
                                                   (L, 23, 22, 3, 16), (S, 25, 26, 3, 16), (L, 27, 30, 8, 16),
                                                   (S, 28, 32, 8, 16), (L, 28, 32, 8, 16), (S, 29, 34, 8, 16)])
def test_more_instances_sampled_chunks_match_oracle(kind, n, C, count, pieces):
    assert pb.pairings_has_swar(kind, n)
    moduli = pb.pairings_default_moduli(pb.pairings_bound_moduli(kind, n) + 1)
    chunks = seeds.sample_chunks(C, count, salt=300 + n)
    want = oracle_rows(kind, n, C, chunks, moduli, threads=16, pieces=pieces)
    for c, w in zip(chunks, want):
        b = min(c & ~31, (1 << C) - 32) if C >= 5 else 0
        e = min(b + 32, 1 << C)
        rows, nz = gpu_rows(kind, n, C, b, e, moduli, pb.LaunchOpts(variant=pb.VARIANT_SWAR), count_nonzero=False), None
        assert rows[c - b] == w[2], (kind, n, c)
        assert pb.pairings_crt_signed(moduli, rows[c - b]) == w[0]


@pytest.mark.parametrize("kind,n", [(S, 9), (L, 15), (S, 17), (L, 19)])
def test_more_paper_totals(kind, n, paper_counts):
    # PAPER.md:349 (S(9)), :352 (S(17)), :377 (L(15)), :379 (L(19))
    full = pb.count(kind, n)
    assert full[1] == paper_counts[(kind, n)] and full[0] == 2 * full[1]
    assert pb.count(kind, n, lemma24=True, duplicate=True) == full


# ---- the chunk farm on one GPU
def test_slices_of_two_jobs_merge_to_the_count(tmp_path, paper_counts):
    kind, n, C = S, 16, 10
    moduli = pb.pairings_default_moduli(pb.pairings_bound_moduli(kind, n) + 1)
    paths = []
    for r in range(3):                                   # three jobs over the x_2 = +1 half (symmetry 3), audited
        b, e = pb.pairings_rank_range(C - 1, r, 3)
        path = str(tmp_path / ("job%d.txt" % r))
        total, done, needed = pb.pairings_run_slice(kind, n, C, moduli, 100, b, e, path, 0, 0, None, pb.RUN_LEMMA24 | pb.RUN_AUDIT)
        assert done == needed == e - b and pb.pairings_run_slice.last_mismatches == 0
        with pytest.raises(pb.PairingsError):            # the journal of one job is not another job's
            pb.pairings_run_slice(kind, n, C, moduli, 100, e % (1 << (C - 1)), (e % (1 << (C - 1))) + 1, path, 0, 0, None, pb.RUN_LEMMA24)
        paths.append(path)
    nr, total, covered = pb.pairings_journal_merge(paths, kind, n, C, moduli)
    assert covered == 1 << (C - 1)
    total = pb.pairings_sum_rows([total], moduli, total)                 # H = 2 x (the x_2 = +1 half)
    assert pb.pairings_reconstruct(kind, n, moduli, total) == (2 * paper_counts[(kind, n)], paper_counts[(kind, n)])
    # the command line does the same: two jobs, then --merge
    from paper_1507_00315_b200 import __main__ as cli
    js = [str(tmp_path / ("cli%d.txt" % r)) for r in range(2)]
    for r in range(2):
        assert cli.main(["L", "12", "--chunk-bits", "6", "--rank", str(r), "--world", "2", "--journal", js[r], "--audit"]) == 0
    assert cli.main(["L", "12", "--chunk-bits", "6", "--merge"] + js) == 0


@pytest.mark.parametrize("extra", [[], ["--lemma24"], ["--lemma24", "--duplicate", "--audit"], ["--lemma24", "--rank", "0", "--world", "1"]])
def test_command_line_prints_the_papers_count(extra, capsys):
    import json
    from paper_1507_00315_b200 import __main__ as cli
    assert cli.main(["S", "16", "--json"] + extra) == 0
    out = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    assert (out["identified"], out["distinct"]) == (700078384, 1400156768)          # PAPER.md:352 (Table 7)
    assert out["chunks_done"] == out["chunks_needed"] == (out["chunks"] // 2 if extra else out["chunks"])
    # a whole run through the slice driver leaves the symmetry factor to the caller: raw sum = half of H
    moduli = pb.pairings_default_moduli(pb.pairings_bound_moduli(S, 16) + 1)
    raw, done, needed = pb.pairings_run_slice(S, 16, 8, moduli, 64, 0, 256, None, 0, 0, None, pb.RUN_LEMMA24)
    full, fdone, fneeded = pb.pairings_run_ex(S, 16, 8, moduli, 64, None, 0, 0, None, pb.RUN_LEMMA24)
    assert done == needed == fdone == fneeded == 128 and pb.pairings_sum_rows([raw], moduli, raw) == full


@pytest.mark.parametrize("kind,n,C", [(L, 12, 6), (S, 13, 8), (L, 16, 10)])
def test_generic_kernel_audits_the_fast_kernel(kind, n, C, paper_counts):
    moduli = pb.pairings_default_moduli(pb.pairings_bound_moduli(kind, n) + 1)
    total, done, needed = pb.pairings_run_ex(kind, n, C, moduli, 1 << (C - 3), None, 0, 0, None, pb.RUN_AUDIT | pb.RUN_DUPLICATE)
    assert done == needed == 1 << C and pb.pairings_run_ex.last_mismatches == 0
    assert pb.pairings_reconstruct(kind, n, moduli, total)[1] == paper_counts[(kind, n)]


def test_bench_self_spawn_path_on_one_gpu():
    import json, os, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "1", "--spawn", "--steps", "1", "--no-cpu", "--no-pt",
                          "--no-configs", "--no-n24"], capture_output=True, text=True, timeout=900, cwd=root, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads([ln for ln in out.stdout.splitlines() if ln.strip()][-1])
    assert d["n_gpus"] == 1 and d["config"]["launcher"] == "self-spawned ranks" and d["scaling"] == "strong" and d["value"] > 1e11


@pytest.mark.parametrize("scaling", ["strong", "duplicate"])
def test_bench_two_ranks_on_two_gpus(scaling):
    """bench.py's N > 1 branch on real devices (NCCL rendezvous, disjoint chunk ranges or the duplicate-run check,
    exchange of the residue sums, max-over-ranks times).  Needs two GPUs: skipped on the one-GPU boxes this repository
    has been developed on — the same exchange code runs under gloo in tests/test_multirank_cpu.py."""
    import json
    import os
    import subprocess
    import sys
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "1", "--no-cpu", "--no-pt",
                          "--no-configs", "--no-n24", "--scaling", scaling], capture_output=True, text=True, timeout=900, cwd=root,
                         env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads([ln for ln in out.stdout.splitlines() if ln.strip()][-1])
    # L(20) was reconstructed from the exchanged sums inside the run (bench asserts it); every sign vector counted once
    assert d["n_gpus"] == 2 and d["scaling"] == ("strong" if scaling == "strong" else "weak") and d["value"] > 1e11

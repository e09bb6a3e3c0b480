"""N > 1 host path on CPU (gloo, world_size 2): each rank owns a contiguous chunk range
(pairings_rank_range), sums its rows, the per-rank sums are exchanged and rank 0 reconstructs.
The rows themselves come from the CPU oracle here (no GPU on this box); on the GPU box bench.py runs
the same exchange around count_pairings."""
import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, kind, n, C, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    import paper_1507_00315_b200 as pb
    moduli = pb.pairings_default_moduli(pb.pairings_min_moduli(kind, n) + 1)
    b, e = pb.pairings_rank_range(C, rank, world)
    rows = [oracle.chunk(kind, n, C, c, moduli)[2] for c in range(b, e)]
    mine = pb.pairings_sum_rows(rows, moduli)
    import bench                                   # bench.py's OWN exchange and time reduction, on gloo instead of NCCL
    total = bench.exchange_sums(dist, mine, moduli, world, False, "cpu", pb.pairings_sum_rows)
    # duplicate-run mode: every rank holds the whole sum, the copies are compared
    same = bench.exchange_sums(dist, total, moduli, world, True, "cpu", pb.pairings_sum_rows)
    slowest = bench.max_over_ranks(dist, 10.0 + rank, "cpu")
    disagree = False
    try:                                           # a rank with another sum must be noticed by every rank
        bench.exchange_sums(dist, [(v + (rank == world - 1)) % p for v, p in zip(total, moduli)], moduli, world, True, "cpu",
                            pb.pairings_sum_rows)
    except AssertionError:
        disagree = True
    if rank == 0:
        q.put((b, e, pb.pairings_reconstruct(kind, n, moduli, total), same == total, slowest, disagree))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("kind,n,C,world,want", [(1, 8, 4, 2, (300, 150)), (0, 9, 5, 2, (2656, 1328)), (0, 7, 3, 2, (0, 0)),
                                                 (1, 8, 4, 3, (300, 150))])
def test_ranks_take_disjoint_ranges_then_bench_exchange_then_crt(kind, n, C, world, want):
    from paper_1507_00315_b200 import build as pbuild
    pbuild.build()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, kind, n, C, q)) for r in range(world)]
    [p.start() for p in procs]
    b, e, got, same, slowest, disagree = q.get(timeout=180)
    [p.join(timeout=120) for p in procs]
    assert all(p.exitcode == 0 for p in procs)
    import paper_1507_00315_b200 as pb
    assert (b, e) == tuple(pb.pairings_rank_range(C, 0, world)) and b == 0 and 0 < e <= -(-(1 << C) // world)
    assert got == want          # L(8)=150, S(9)=1,328, S(7): no pairing
    assert same and disagree and slowest == 10.0 + world - 1


def test_cli_merges_two_rank_journals_of_L12(tmp_path, capsys):
    """The paper's workflow: N independent jobs, results put together afterwards.  Here the rows
    of each rank's slice come from the CPU oracle (no GPU on this box); the journals, the merge and the CLI are the
    product's.  L(12) = 108,144.  With symmetry 3 only the x_2 = +1 half is dealt out and doubled."""
    import json
    import threading
    import oracle
    import paper_1507_00315_b200 as pb
    from paper_1507_00315_b200 import __main__ as cli
    kind, n, C = pb.LANGFORD, 12, 6
    moduli = pb.pairings_default_moduli(pb.pairings_bound_moduli(kind, n) + 1)
    rows = [None] * (1 << C)

    def work(t):
        for c in range(t, 1 << C, 8):
            rows[c] = oracle.chunk(kind, n, C, c, moduli)[2]
    ts = [threading.Thread(target=work, args=(t,)) for t in range(8)]
    [t.start() for t in ts]
    [t.join() for t in ts]

    def journals(bits, tag):
        paths = []
        for r in range(2):
            b, e = pb.pairings_rank_range(bits, r, 2)
            path = str(tmp_path / ("%s_%d.txt" % (tag, r)))
            for lo in range(b, e, 7):
                hi = min(lo + 7, e)
                pb.pairings_journal_append(path, kind, n, C, moduli, lo, hi, pb.pairings_sum_rows(rows[lo:hi], moduli))
            paths.append(path)
        return paths

    full = journals(C, "full")
    assert cli.main(["L", "12", "--chunk-bits", "6", "--json", "--merge"] + full) == 0
    out = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    assert (out["identified"], out["distinct"], out["chunks_done"]) == (108144, 216288, 64)
    half = journals(C - 1, "half")                                     # symmetry 3: chunks [0, 32) only
    assert cli.main(["L", "12", "--chunk-bits", "6", "--lemma24", "--json", "--journal", str(tmp_path / "m.txt"), "--merge"] + half) == 0
    out = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    assert (out["identified"], out["chunks_done"], out["chunks_needed"]) == (108144, 32, 32)
    assert pb.pairings_journal_load(str(tmp_path / "m.txt"), kind, n, C, moduli)[0][-1][1] == 32
    # one rank missing: incomplete, exit code 3, no count printed
    assert cli.main(["L", "12", "--chunk-bits", "6", "--json", "--merge", full[0]]) == 3
    out = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    assert "identified" not in out and out["chunks_done"] == 32
    # overlapping journals (the same rank twice) and journals of the other mode are refused
    with pytest.raises(pb.PairingsError):
        cli.main(["L", "12", "--chunk-bits", "6", "--merge", full[0], full[0]])

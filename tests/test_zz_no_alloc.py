"""pairings_pt_run_noalloc: the approximate counter for callers that must not allocate device memory.

Some users of this library cannot call cudaMalloc: a server that gave all of HBM to its own arena at start-up, a loop
with a latency budget that an allocator call (which may synchronise the whole device) would break, or a plug-in whose
host application owns the memory budget.  For them the library keeps the one piece of scratch memory the
parallel-tempering kernel needs — its acceptance-threshold table — in a fixed 16 KiB `static __device__` array, and
this entry point uses that instead of cudaMallocAsync.  What has to hold:

  * the counters are bit-identical to pairings_pt_run's (same kernel, integer decisions: tolerance zero, as in
    tests/test_pt_gpu.py), on two calls in a row — the second with a SHORTER ladder and a smaller n, so that anything
    the first call left in the shared array would show up as a difference;
  * a request whose table does not fit the array is refused with PAIRINGS_ETOOBIG and enqueues nothing.

The file sorts last on purpose: the driver runs pytest with -x, and a failure here must not hide the parity tests.
It passes alone in a fresh process (the first call then does the per-device address look-up) and after the others."""
import pytest

import paper_1507_00315_b200 as pb

S, L = pb.SKOLEM, pb.LANGFORD
ETOOBIG = -12


def _counters(entry, kind, n, betas, r0, r1, iterations, burn, seed):
    import torch
    M, N = len(betas), 2 * n
    hist = torch.zeros((M, N + 1), dtype=torch.int64, device="cuda")
    mv = torch.zeros(M, dtype=torch.int64, device="cuda")
    sw = torch.zeros(M, dtype=torch.int64, device="cuda")
    entry(kind, n, betas, r0, r1, iterations, burn, seed, hist.data_ptr(), mv.data_ptr(), sw.data_ptr(),
          torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return hist.cpu().tolist(), mv.cpu().tolist(), sw.cpu().tolist()


@pytest.mark.gpu
def test_noalloc_counters_equal_the_allocating_path_on_two_calls_in_a_row():
    pytest.importorskip("torch")
    calls = [
        # a long ladder at a large n first: 11 x (32 + 3) = 385 words of the shared table
        (L, 16, [0, 0.5, 1.0, 1.6, 2.3, 3.1, 4.0, 5.2, 7.0, 11.0, 20.0], 0, 100, 200, 20, 7),
        # then a short one at a small n: 4 x 11 = 44 words, the other 341 still hold the first call's thresholds
        (L, 4, [0, 1.0, 2.2, 4.0], 3, 103, 300, 17, 2),
        # and the Table 6 ladder, ragged replica count
        (S, 12, [0, 0.54, 1.1, 1.69, 2.33, 3, 3.73, 4.65, 5.82, 8.1, 16, 32], 0, 70, 400, 100, 150700315),
    ]
    got = [_counters(pb.pairings_pt_run_noalloc, *c) for c in calls]          # back to back, nothing in between
    want = [_counters(pb.pairings_pt_run, *c) for c in calls]
    for c, g, w in zip(calls, got, want):
        assert sum(map(sum, w[0])) == (c[4] - c[3]) * (c[5] - c[6]) * len(c[2])   # the existing path did run
        assert g[0] == w[0], c
        assert g[1] == w[1] and g[2] == w[2], c
    # the same call again gives the same counters (the table is rewritten, not accumulated)
    assert _counters(pb.pairings_pt_run_noalloc, *calls[1]) == want[1]


@pytest.mark.gpu
def test_noalloc_adds_to_the_callers_counters_and_takes_an_empty_range():
    torch = pytest.importorskip("torch")
    kind, n, betas = S, 8, [0, 0.8, 1.8, 3.0, 6.0]
    whole = _counters(pb.pairings_pt_run_noalloc, kind, n, betas, 0, 150, 128, 8, 5)
    M, N = len(betas), 2 * n
    hist = torch.zeros((M, N + 1), dtype=torch.int64, device="cuda")
    mv = torch.zeros(M, dtype=torch.int64, device="cuda")
    sw = torch.zeros(M, dtype=torch.int64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    for r0, r1 in ((0, 37), (37, 37), (37, 150)):                            # same stream: ordered, no race on the table
        pb.pairings_pt_run_noalloc(kind, n, betas, r0, r1, 128, 8, 5, hist.data_ptr(), mv.data_ptr(), sw.data_ptr(), st)
    torch.cuda.synchronize()
    assert (hist.cpu().tolist(), mv.cpu().tolist(), sw.cpu().tolist()) == whole
    assert whole == _counters(pb.pairings_pt_run, kind, n, betas, 0, 150, 128, 8, 5)


def test_noalloc_refuses_what_does_not_fit_its_table():
    """No GPU needed: sizes are checked before the first CUDA call.  32 levels at n = 32 need 32 x 67 = 2144 words,
    the array has 2048; 30 levels (2010 words) fit, so that request gets past the size check (and then stops at the
    NULL counters)."""
    betas = [0.25 * j for j in range(32)]
    with pytest.raises(pb.PairingsError) as too_big:
        pb.pairings_pt_run_noalloc(L, 32, betas, 0, 1, 10, 0, 1, 0, 0, 0)
    assert too_big.value.code == ETOOBIG and "no-allocation" in str(too_big.value)
    with pytest.raises(pb.PairingsError) as fits:
        pb.pairings_pt_run_noalloc(L, 32, betas[:30], 0, 1, 10, 0, 1, 0, 0, 0)
    assert fits.value.code == -5                                               # PAIRINGS_ENULL, not ETOOBIG
    with pytest.raises(pb.PairingsError) as bad:
        pb.pairings_pt_run_noalloc(L, 32, [0.5, 1.0], 0, 1, 10, 0, 1, 0, 0, 0)    # betas[0] must be 0, as in pairings_pt_run
    assert bad.value.code == -10


def test_noalloc_entry_point_names_no_allocating_call():
    """A source-level guard for the promise in the header: between its opening brace and the next top-level function,
    pairings_pt_run_noalloc (and the address look-up it uses) must not mention cudaMalloc*, cudaFree*, a memory pool or
    a std::vector, and the look-up must go through cudaGetSymbolAddress with its return code checked."""
    import os
    import re
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    src = open(os.path.join(root, "paper_1507_00315_b200", "csrc", "pt_kernel.cu")).read()
    src = re.sub(r"//[^\n]*", "", src)                                        # comments may name what is avoided
    body = src[src.index("int pairings_pt_run_noalloc("):]
    body = body[:body.index("\nint pairings_pt_ladder(")]
    lookup = src[src.index("static int pt_static_address("):]
    lookup = lookup[:lookup.index("\n}\n") + 3]
    for text in (body, lookup):
        for banned in ("cudaMalloc", "cudaFree", "cudaMemPool", "cudaHostAlloc", "std::vector", "new ", "malloc("):
            assert banned not in text, banned
    assert "pt_static_address(&table)" in body and "PAIRINGS_ETOOBIG" in body
    assert re.search(r"cudaGetSymbolAddress\(&ptr, pt_static_thr\)", lookup) and "e != cudaSuccess" in lookup
    assert re.search(r"static __device__ __align__\(256\) unsigned long long pt_static_thr\[PAIRINGS_PT_STATIC_WORDS\]", src)

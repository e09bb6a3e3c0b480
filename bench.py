#!/usr/bin/env python
"""bench.py — Godfrey sign-vector terms/s on B200 (BASELINE.json metric), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

A "step" is one pass of the whole hot path over the workload: partition -> count_pairings (the
Gray-code kernel over every chunk of this rank's range) -> rows D2H -> row sums -> (rank 0, after
the exchange of the per-rank sums) CRT + exact division, checked against the paper's printed count.
Workload at every N: Langford L(20) — 2^39 sign vectors (x_1 = +1), 2^16 prefix chunks, 6 CRT primes
+ 1 check prime (BASELINE.json configs[3], the n = 20 point the metric is quoted on).

N > 1: the path shards by chunk ranges with no data-path collective ("split ... into several
independent sets and simply put the result together at the end").  `--gpus N` starts the N ranks itself when it is not
already running under torchrun (WORLD_SIZE unset): N copies of this script with RANK / LOCAL_RANK / WORLD_SIZE /
MASTER_ADDR=127.0.0.1 / MASTER_PORT set, one GPU each, NCCL for the barrier and the exchange of the per-rank residue
sums.  Under torchrun WORLD_SIZE must equal --gpus.  The ranks take DISJOINT chunk ranges (pairings_rank_range; total
work fixed: "scaling": "strong"), their sums are added and L(20) is reconstructed from them.  `--scaling duplicate`
(opt-in) is the paper's duplicate-run check: every rank evaluates the whole pass, the copies must agree;
its `value` counts the sign vectors ONCE.

`value`   = terms/s with the rows left in HBM (CUDA events around the kernel launches of a step).
`e2e`     = terms/s through count_pairings_host (HOST output buffer; allocation, launch, D2H copy
            and synchronise inside the timed region, wall clock).
`roofline`= `frac` = issue-slot fraction: EXECUTED thread-instructions per term of the profiled kernel
            (profiles/ncu_metrics.json, ignored when the kernel source changed since the capture) x terms/s measured
            here, against the SM integer-issue peak 148 x 128 lanes x sm_max_mhz.  Beside it `useful_frac` (the minimum
            instruction count of the design as built, same rate and peak), `yardstick_frac` (SURVEY.md
            §8(d)'s fixed model W + phi*M of a scalar kernel: a speed-up over that design, not a utilisation) and
            `n24`, the S(24) point of the metric with its own fractions and clocks.
`cpu_baseline` = the CPU oracle (oracle/, as it stands) on the host cores, bounded sample, all cores and 1 core.
"""
from __future__ import annotations

import argparse
import ctypes
import json
import os
import socket
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

KIND_NAME = {0: "S", 1: "L"}
# workload (BASELINE.json configs[3]): Langford n = 20, 2^16 chunks, 6 primes + 1 check prime
WL = dict(kind=1, n=20, chunk_bits=16, n_moduli=7)
L20_IDENTIFIED = 2636337861200          # L(20), PAPER.md:380 (Table 8)
WORKLOAD = "L(20): Langford n=20, 2^39 sign vectors (x_1=+1), 2^16 prefix chunks, 6 CRT primes + 1 check prime, full count per step"
# secondary point of the metric (configs[4]): Skolem n = 24, 2^20 chunks, 8 primes + 1 check prime,
# a fixed seeded 1/64 subset of chunks (16 runs of 1024 contiguous chunks: launches long enough that the last,
# partly filled wave of blocks does not dominate)
WL24 = dict(kind=0, n=24, chunk_bits=20, n_moduli=9, runs=16, run_len=1024)
# BASELINE.json configs[0..3] other than the workload: (kind, n, chunk_bits, moduli incl. check, back-to-back
# launches timed, printed count: PAPER.md Table 8 :376,:378 / Table 7 :351,:352,:354)
OTHER_CONFIGS = [(1, 12, 6, 4, 100, 108144), (0, 13, 8, 4, 100, 1520280), (1, 16, 10, 6, 20, 326721800),
                 (0, 16, 10, 6, 20, 700078384), (0, 21, 18, 7, 1, 61782464083584)]
PT_BETAS = [0, 0.54, 1.1, 1.69, 2.33, 3, 3.73, 4.65, 5.82, 8.1, 16, 32]     # PAPER.md:329-341 (Table 6, column beta)
SM_COUNT, LANES_PER_SM_CLK = 148, 128
NCU_METRICS = os.path.join(ROOT, "profiles", "ncu_metrics.json")


def yardstick_ops(kind: int, n: int, n_moduli: int, phi: float):
    """ops(kind,n,m') = W + phi*M, W = 3n+3, M = (n-G) + m'(5(G-1)+3), G = greedy
    grouping of the factor bounds 2n-d_k into exact <= 31-bit partial products."""
    bounds = [2 * n - (k if kind == 0 else k + 1) for k in range(1, n + 1)]
    G, prod = 1, 1
    for b in bounds:
        if prod * b >= 1 << 31:
            G, prod = G + 1, 1
        prod *= b
    W = 3 * n + 3
    M = (n - G) + n_moduli * (5 * (G - 1) + 3)
    return W + phi * M, dict(W=W, M=M, G=G, phi=phi)


KERNEL_SOURCES = {"instances": ["swar_kernel.cuh", "device_common.cuh"], "pt": ["pt_kernel.cu"]}


def kernel_source_sha16(which: str) -> str:
    """sha256 (16 hex digits) over the source files of a profiled kernel — recorded with every ncu capture in
    profiles/ncu_metrics.json, so that a capture of an older kernel is recognised without git (the GPU box has none)."""
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES[which]:
        with open(os.path.join(ROOT, "paper_1507_00315_b200", "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def ncu_record(which: str, key=None):
    """(record, stale) — the ncu capture of a kernel from profiles/ncu_metrics.json (`which` = "instances" with key
    "L20", or "pt"); stale = the kernel's source files no longer hash to what the capture recorded.  (None, False)
    when there is no record."""
    try:
        with open(NCU_METRICS) as f:
            doc = json.load(f)
        rec = doc[which] if key is None else doc[which].get(key)
    except (OSError, ValueError, KeyError):
        return None, False
    if not rec:
        return None, False
    return rec, rec.get("source_sha16") != kernel_source_sha16(which)


def swar_plan(kind: int, n: int):
    """The packed-sum layout and product plan of swar_kernel<kind, n> (csrc/swar_kernel.cuh, Lay::make_plan), restated
    for the instruction accounting: NR packed registers, E even distances, pair / single factors, G groups with exact
    products below 2^31 (best fit decreasing), W accumulator words."""
    N = 2 * n
    ds = [k if kind == 0 else k + 1 for k in range(1, n + 1)]
    slots = [d for d in ds if d % 2 == 0] + [d for d in ds if d % 2 == 1]
    bound = [((N - d) // 2 if d % 2 == 0 else N - d) for d in slots]
    NR = (n + 3) // 4
    sb = lambda s: bound[s] if s < n else 0

    def plan(last_as_singles):
        fac = []                                            # (bound, is_pair)
        for pp in range(NR // 2):
            r = 2 * pp
            for i in range(4):
                b1, b2 = sb(4 * r + i), sb(4 * (r + 1) + i)
                if b1 and b2:
                    fac.append((b1 * b2, True))
                elif b1:
                    fac.append((b1, False))
        if NR % 2 == 1:
            r = NR - 1
            for i in range(0, 4, 1 if last_as_singles else 2):
                b1, b2 = sb(4 * r + i), 0 if last_as_singles else sb(4 * r + i + 1)
                if b1 and b2:
                    fac.append((b1 * b2, True))
                elif b1:
                    fac.append((b1, False))
        order = sorted(range(len(fac)), key=lambda f: -fac[f][0])
        for G in range(1, 9):
            prod, ok = [1] * G, True
            for f in order:
                best = -1
                for g in range(G):
                    if prod[g] * fac[f][0] < 1 << 31 and (best < 0 or prod[g] > prod[best]):
                        best = g
                if best < 0:
                    ok = False
                    break
                prod[best] *= fac[f][0]
            if ok:
                bits = sum(p.bit_length() for p in prod)
                return dict(G=G, W=(bits + 33 + 31) // 32, nf=len(fac), pairs=sum(1 for f in fac if f[1]),
                            singles=sum(1 for f in fac if not f[1]))
        raise ValueError("no grouping")

    a, b = plan(True), plan(False)
    best = a if a["G"] < b["G"] else b
    best.update(NR=NR, E=sum(1 for d in ds if d % 2 == 0))
    return best


def useful_instr(kind: int, n: int, phi: float):
    """Minimum thread-instructions per term of the SWAR design AS BUILT — the method's arithmetic
    only, no compaction, no loop or address overhead (O(n) additions and multiplications per Gray step):
      every step        NR packed adds (the n byte sums in NR registers) + 4 E / 32 for the zero test (4 instructions
                        per even distance and 32-step block: table address, load, OR, predicate extraction)
      non-zero (x phi)  NR un-bias XORs, 2 per pair factor (operand isolation + IDP.4A) and 1 per single, one 32-bit
                        multiply per factor into its group, 2 for the sign, wide(G) for the exact multi-word product
                        (G = 1: 0, 2: 1, 3: 5, 4: 10 IMAD.WIDE / digit splits; G >= 5: G(G-1)/2 + G + W + 2),
                        W add-with-carry into the accumulator."""
    pl = swar_plan(kind, n)
    G, W = pl["G"], pl["W"]
    wide = {1: 0, 2: 1, 3: 5, 4: 10}.get(G, G * (G - 1) // 2 + G + W + 2)
    per_step = pl["NR"] + 4.0 * pl["E"] / 32
    per_nonzero = pl["NR"] + 2 * pl["pairs"] + pl["singles"] + pl["nf"] + 2 + wide + W
    return per_step + phi * per_nonzero, dict(plan=pl, per_step=per_step, per_nonzero_term=per_nonzero, phi=phi)


def roofline_object(kind, n, n_moduli, phi, terms_per_launch, kernel_s, peak_mhz):
    """`frac` = executed thread-instructions (ncu capture of this kernel instance) x terms/s (measured here) / issue
    peak; `useful_frac` = the design's minimum instruction count at the same rate; `yardstick_frac` = SURVEY §8(d)'s
    model of a scalar kernel (> 1 here: the kernel needs fewer instructions than that model, it skips no work)."""
    ops, ys = yardstick_ops(kind, n, n_moduli, phi)
    peak = SM_COUNT * LANES_PER_SM_CLK * peak_mhz * 1e6
    rate = terms_per_launch / kernel_s
    useful, ud = useful_instr(kind, n, phi)
    r = dict(bound="alu", achieved=None, peak=peak / 1e12, unit="Tinstr/s", frac=None, traffic=None,
             peak_source="formula: 148 SM x 128 lanes/clk x %.0f MHz (clocks.max.sm); MEASURED_PEAKS.json has no integer figure" % peak_mhz,
             kernel_ms=kernel_s * 1e3, terms_per_launch=terms_per_launch, terms_per_s=rate,
             useful_instr_per_term=useful, useful_frac=useful * rate / peak, useful_model=ud,
             ops_per_term=ops, yardstick=ys, yardstick_frac=ops * rate / peak,
             frac_note="frac = executed thread-instructions per term (ncu) x terms/s (CUDA events, this run) / peak: issue slots busy. "
                       "useful_frac = minimum instruction count of the design as built (DESIGN.md 4.3) at the same rate: issue slots "
                       "doing Godfrey arithmetic. yardstick_frac = SURVEY 8(d)'s fixed model of a scalar per-term-Montgomery kernel, "
                       "> 1 because this kernel needs fewer instructions than that model (packed sums, table-driven zero test, "
                       "residues once per thread); the count is reconstructed and checked in every run")
    m, stale = ncu_record("instances", "%s%d" % (KIND_NAME[kind], n))
    if m and not stale:
        r.update(executed_instr_per_term=m["instr_per_term"], achieved=m["instr_per_term"] * rate / 1e12,
                 frac=m["instr_per_term"] * rate / peak, issue_active_pct=m["issue_active_pct"], ncu_source=m.get("source"),
                 ncu_commit=m.get("commit"), ncu_source_sha16=m.get("source_sha16"), traffic=m.get("dram_bytes_per_launch"))
    elif m:
        r.update(ncu_stale=True, ncu_commit=m.get("commit"),
                 ncu_note="the kernel source changed since the ncu capture in profiles/ncu_metrics.json: no executed-instruction "
                          "figure is claimed for this build (frac = null); useful_frac and yardstick_frac need no capture")
    return r


def exchange_sums(dist, total, moduli, world, duplicate, device, sum_rows):
    """The ONE exchange of the N > 1 path ("simply put the result together at the end"): every rank's
    residue sums are gathered and added modulo the primes (disjoint ranges), or compared (duplicate-run check,
    PAPER.md:99).  `dist` = torch.distributed with an initialised default group (NCCL on GPUs, gloo in the CPU tests);
    `sum_rows(rows, moduli)` = pairings_sum_rows.  Returns the job's residue sums on every rank."""
    import torch
    t = torch.tensor(total, dtype=torch.int64, device=device)
    gathered = [torch.zeros_like(t) for _ in range(world)]
    dist.all_gather(gathered, t)
    if duplicate:                                    # every rank counted everything: the copies must agree
        assert all(g.tolist() == list(total) for g in gathered), "ranks disagree (PAPER.md:99 duplicate-run check)"
        return list(total)
    return sum_rows([g.tolist() for g in gathered], moduli)


def max_over_ranks(dist, x: float, device) -> float:
    """A time is the slowest rank's."""
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def host_threads() -> int:
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:
        return os.cpu_count() or 1


# ------------------------------------------------------------------------------------------------
# CPU oracle timing (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------------
def oracle_sample(kind, n, sample_bits, chunks, threads):
    """Times oracle.chunk on `chunks` (indices of the 2^sample_bits partition) with `threads` host
    threads (ctypes releases the GIL).  Returns (terms, seconds)."""
    import oracle
    oracle.build()
    moduli = []
    todo = list(chunks)
    lock = threading.Lock()

    def work():
        while True:
            with lock:
                if not todo:
                    return
                c = todo.pop()
            oracle.chunk(kind, n, sample_bits, c, moduli)

    t0 = time.perf_counter()
    ts = [threading.Thread(target=work) for _ in range(threads)]
    [t.start() for t in ts]
    [t.join() for t in ts]
    dt = time.perf_counter() - t0
    terms = len(chunks) * (1 << (2 * n - 1 - sample_bits))
    return terms, dt


def cpu_baseline(kind, n, target_seconds=12.0):
    from paper_1507_00315_b200 import seeds
    threads = host_threads()
    sample_bits = 2 * n - 1 - 17                       # 2^17 terms per oracle chunk
    probe = seeds.sample_chunks(sample_bits, threads, salt=7)
    terms, dt = oracle_sample(kind, n, sample_bits, probe, threads)
    rate = terms / dt
    count = int(max(threads, min(4096, target_seconds * rate / (1 << 17))))
    chunks = seeds.sample_chunks(sample_bits, count, salt=11)
    terms, dt = oracle_sample(kind, n, sample_bits, chunks, threads)
    # one core ("report terms/s for 1 core and all cores"): ~4 s of the same kind of chunks
    one = seeds.sample_chunks(sample_bits, int(max(2, min(512, 4.0 * rate / threads / (1 << 17)))), salt=13)
    terms1, dt1 = oracle_sample(kind, n, sample_bits, one, 1)
    return dict(value=terms / dt, unit="terms/s", cores=threads, kind="oracle", value_1core=terms1 / dt1,
                sample="%d seeded chunks of 2^17 sign vectors of %s(%d) (2^%d-chunk partition of the x_1=+1 half), "
                       "%.1f s on %d threads; 1 core: %d such chunks, %.1f s" %
                       (len(chunks), KIND_NAME[kind], n, sample_bits, dt, threads, len(one), dt1))


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_1507_00315_b200 import seeds
    kind, n = WL["kind"], WL["n"]
    threads = host_threads()
    sample_bits = 2 * n - 1 - 17
    per_step = 16 * threads
    steps, warm = args.steps, args.warmup
    for w in range(warm):
        oracle_sample(kind, n, sample_bits, seeds.sample_chunks(sample_bits, threads, salt=100 + w), threads)
    terms_total, t_total = 0, 0.0
    for s in range(steps):
        terms, dt = oracle_sample(kind, n, sample_bits, seeds.sample_chunks(sample_bits, per_step, salt=200 + s), threads)
        terms_total += terms
        t_total += dt
    value = terms_total / t_total
    sample = "%d seeded chunks of 2^17 sign vectors of L(20) per step on %d threads" % (per_step, threads)
    line = dict(impl="reference", metric="godfrey_sign_vector_terms_per_s", value=value, unit="terms/s",
                n_gpus=args.gpus, steps=steps, warmup=warm, ms_per_step=1e3 * t_total / steps,
                higher_is_better=True, scaling="strong", vs_baseline=None, dtype="int32", data="synthetic",
                config=dict(workload=WORKLOAD, kind="langford", n=n, chunk_bits=WL["chunk_bits"], n_moduli=WL["n_moduli"]),
                cpu_baseline=dict(value=value, unit="terms/s", cores=threads, kind="oracle",
                                  sample="each step is a bounded sample of the workload: " + sample),
                e2e=dict(value=value, unit="terms/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                gpu_launches=0)
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
# clocks
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append((time.perf_counter(), ln.strip()))

    def close(self):
        if self.proc is not None:
            self.proc.terminate()

    def window(self, t0, t1):
        """Clock statistics of the samples taken in [t0, t1] (the sampler keeps running: starting nvidia-smi
        inside or right before a wall-clock region would perturb it)."""
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.25)
        sm, mx, power, reasons = [], None, [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for t, ln in self.lines:
            if t < t0 or t > t1 + 0.3:
                continue
            f = [x.strip() for x in ln.split(",")]
            try:
                sm.append(float(f[0]))
                mx = float(f[1])
                power.append(float(f[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return dict(sm_mhz=statistics.median(sm) if sm else None, sm_max_mhz=mx, samples=len(sm),
                    power_w_max=max(power) if power else None, reasons=sorted(reasons))


_probe_lib = None


def issue_probe(mode, blocks, threads, iters, out_dev_ptr, stream):
    """Enqueues a calibration kernel of libpairings_probe.so (bench-side, not in the product library); returns the
    number of thread-instructions it executes."""
    global _probe_lib
    if _probe_lib is None:
        from paper_1507_00315_b200 import build as pbuild
        _probe_lib = ctypes.CDLL(pbuild.build_probe())
        _probe_lib.pairings_issue_probe.restype = ctypes.c_int
        _probe_lib.pairings_issue_probe.argtypes = [ctypes.c_int] * 4 + [ctypes.c_void_p, ctypes.c_void_p, ctypes.POINTER(ctypes.c_uint64)]
    cnt = ctypes.c_uint64(0)
    rc = _probe_lib.pairings_issue_probe(mode, blocks, threads, iters, ctypes.c_void_p(out_dev_ptr), ctypes.c_void_p(stream), ctypes.byref(cnt))
    if rc:
        raise RuntimeError("pairings_issue_probe failed: %d" % rc)
    return int(cnt.value)


# ------------------------------------------------------------------------------------------------
# GPU arm
# ------------------------------------------------------------------------------------------------
def run_gpu(args):
    import torch
    import paper_1507_00315_b200 as pb
    from paper_1507_00315_b200 import seeds

    from paper_1507_00315_b200 import build as pbuild
    if not os.path.exists(pb.library_path()):
        pbuild.build()                         # fresh checkout: build in-tree (nvcc, sm_100a)
    pb.lib()                                   # fails loudly if the CUDA library is missing
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d (start it as `python bench.py --gpus N`, which spawns the ranks "
                         "itself, or under torchrun with --nproc-per-node equal to --gpus)" % (args.gpus, world))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    if local >= torch.cuda.device_count():
        raise SystemExit("bench.py: rank %d needs cuda:%d but only %d device(s) are visible" % (rank, local, torch.cuda.device_count()))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    kind, n, C, m = WL["kind"], WL["n"], WL["chunk_bits"], WL["n_moduli"]
    moduli = pb.pairings_default_moduli(m)
    duplicate = args.scaling == "duplicate"
    begin, end = (0, 1 << C) if duplicate else pb.pairings_rank_range(C, rank, world)
    if args.profile_chunks:                      # short launches for ncu captures; not a bench value
        end = min(end, begin + args.profile_chunks)
    rows = end - begin
    terms_rank = rows << (2 * n - 1 - C)
    # sign vectors of the JOB, each counted once (duplicate mode: N copies of the same pass are one pass)
    terms_job = terms_rank * (1 if duplicate else world) if args.profile_chunks else (1 << (2 * n - 1))
    stream = torch.cuda.current_stream().cuda_stream
    out = torch.empty((rows, m), dtype=torch.int32, device="cuda")
    host_rows = torch.empty((rows, m), dtype=torch.int32).pin_memory()
    host_ptr = ctypes.cast(host_rows.data_ptr(), ctypes.POINTER(ctypes.c_uint32))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2

    def launch_opts(nonzero_ptr=None):
        o = pb.LaunchOpts(variant=pb.VARIANT_AUTO, gray_bits=0, block_threads=0, blocks_per_chunk=0)   # library defaults
        if nonzero_ptr is not None:
            o.nonzero_terms = nonzero_ptr
        return o

    opts = launch_opts()
    geometry = pb.pairings_query_geometry(kind, n, C, rows, opts)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step_device():
        pb.count_pairings_ex(kind, n, C, begin, end, moduli, out.data_ptr(), stream, opts)

    def finish(rows_tensor):
        """rows -> per-rank sum -> exchange -> CRT on rank 0 (outside the timed region for `value`)."""
        flat = (ctypes.c_uint32 * (rows * m)).from_address(rows_tensor.data_ptr())
        total = pb.pairings_sum_rows(flat, moduli)
        if dist is not None:
            total = exchange_sums(dist, total, moduli, world, duplicate, "cuda", pb.pairings_sum_rows)
        if rank == 0 and not args.profile_chunks:
            D, S = pb.pairings_reconstruct(kind, n, moduli, total)
            assert S == L20_IDENTIFIED and D == 2 * S, ("L(20) mismatch", D, S)
        return total

    sampler = ClockSampler(local)          # one nvidia-smi for the whole run, started well before the timed regions
    sampler.start()

    # ---- warm-up (>= 3), correctness of the warmed-up path
    warm = max(args.warmup, 3)
    for _ in range(warm):
        step_device()
        flush.fill_(1)
    torch.cuda.synchronize()
    host_rows.copy_(out)
    finish(host_rows)

    # ---- phi (exact non-zero fraction) from the kernel's own counter, untimed
    nzt = torch.zeros(1, dtype=torch.int64, device="cuda")
    pb.count_pairings_ex(kind, n, C, begin, end, moduli, out.data_ptr(), stream, launch_opts(nzt.data_ptr()))
    torch.cuda.synchronize()
    phi = float(nzt.item()) / terms_rank

    # ---- timed: K steps, CUDA events per step on the launching stream, L2 flushed between steps
    barrier()
    t_begin = time.perf_counter()
    evs = []
    for _ in range(args.steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        step_device()
        e1.record()
        evs.append((e0, e1))
        flush.fill_(1)
    barrier()
    t_end = time.perf_counter()
    clocks = sampler.window(t_begin, t_end)
    dev_ms = sum(a.elapsed_time(b) for a, b in evs)
    rank_kernel_s = dev_ms * 1e-3 / args.steps            # this rank's kernel
    if dist is not None:
        dev_ms = max_over_ranks(dist, dev_ms, "cuda")
    launches = (warm + 1 + args.steps) * world  # one kernel launch per pass and rank (grid = chunks of the rank)
    value = terms_job * args.steps / (dev_ms * 1e-3)

    # ---- e2e: the public host-buffer call, wall clock, copies + allocation inside
    for _ in range(2):
        pb.count_pairings_host(kind, n, C, begin, end, moduli, stream, opts, out=host_ptr)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        pb.count_pairings_host(kind, n, C, begin, end, moduli, stream, opts, out=host_ptr)
        finish(host_rows)
    barrier()
    e2e_s = time.perf_counter() - t0
    clocks_e2e = sampler.window(t0, t0 + e2e_s)
    if dist is not None:
        e2e_s = max_over_ranks(dist, e2e_s, "cuda")
    e2e_value = terms_job * args.steps / e2e_s
    launches += (2 + args.steps) * world

    extras = rank == 0 and world == 1 and not args.profile_chunks      # the single-GPU side measurements
    # ---- whole count with symmetry 3 (Lemma 2.4, §8(f) NEXT #1): half the chunks, doubled; wall clock, rank 0
    lemma24 = None
    if extras:
        t0 = time.perf_counter()
        tot, done, needed = pb.pairings_run_ex(kind, n, C, moduli, 1 << C, None, 0, stream, opts, pb.RUN_LEMMA24)
        dt = time.perf_counter() - t0
        D, S = pb.pairings_reconstruct(kind, n, moduli, tot)
        assert S == L20_IDENTIFIED and done == needed == 1 << (C - 1)
        lemma24 = dict(seconds=dt, chunks_evaluated=needed, terms_evaluated=needed << (2 * n - 1 - C),
                       note="pairings_run_ex(PAIRINGS_RUN_LEMMA24): x_2 = +1 half of the chunks, doubled; same count")
        launches += 1

    line = None
    if rank == 0:
        peak_mhz = clocks.get("sm_max_mhz") or 1965.0
        peak = SM_COUNT * LANES_PER_SM_CLK * peak_mhz * 1e6
        roofline = roofline_object(kind, n, m, phi, terms_rank, rank_kernel_s, peak_mhz)
        # calibration kernels: measured thread-instr/s per instruction class
        cal = {}
        scratch = torch.zeros(4, dtype=torch.int32, device="cuda")
        for mode, name in ((0, "iadd3"), (1, "lop3"), (2, "imad"), (3, "iadd3_imad_1to1")):
            best = 0.0
            for rep in range(3):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                cnt = issue_probe(mode, SM_COUNT * 8, 256, 4096, scratch.data_ptr(), stream)
                e1.record()
                torch.cuda.synchronize()
                best = max(best, cnt / (e0.elapsed_time(e1) * 1e-3))
            cal[name] = best / 1e12
        roofline["calibration_Tinstr_per_s"] = cal
        if roofline["achieved"] is not None:       # against the best measured instruction mix instead of the formula peak
            roofline["frac_of_best_calibration"] = roofline["achieved"] / max(cal.values())

        # secondary point of the metric: S(24) on the seeded 1/64 subset (BASELINE.json configs[4])
        n24 = None
        if not args.no_n24 and world == 1:
            k2, n2, C2, m2 = WL24["kind"], WL24["n"], WL24["chunk_bits"], WL24["n_moduli"]
            mod2 = pb.pairings_default_moduli(m2)
            runs = max(1, int(round(WL24["runs"] * args.n24_fraction)))
            starts = seeds.sample_range_starts(C2, runs, WL24["run_len"])
            out2 = torch.empty((WL24["run_len"], m2), dtype=torch.int32, device="cuda")
            nz24 = torch.zeros(1, dtype=torch.int64, device="cuda")
            o24 = launch_opts(nz24.data_ptr())
            # untimed: every run once with the non-zero counter = warm-up launches (>= 2) and the exact phi of the subset
            warm24 = starts if len(starts) >= 2 else starts * 2
            for s0 in warm24:
                pb.count_pairings_ex(k2, n2, C2, s0, s0 + WL24["run_len"], mod2, out2.data_ptr(), stream, o24)
            torch.cuda.synchronize()
            terms24 = len(starts) * WL24["run_len"] << (2 * n2 - 1 - C2)
            phi24 = float(nz24.item()) / (terms24 * len(warm24) // len(starts))
            flush.fill_(1)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for s0 in starts:
                pb.count_pairings_ex(k2, n2, C2, s0, s0 + WL24["run_len"], mod2, out2.data_ptr(), stream, opts)
            e1.record()
            torch.cuda.synchronize()
            t1 = time.perf_counter()
            t24 = e0.elapsed_time(e1) * 1e-3
            launches += len(warm24) + len(starts)
            n24 = dict(workload="S(24): %d seeded runs of %d contiguous chunks of the 2^20-chunk partition (= 1/%d of the chunks), 8+1 primes"
                                % (len(starts), WL24["run_len"], (1 << C2) // (len(starts) * WL24["run_len"])),
                       terms=terms24, seconds=t24, value=terms24 / t24, unit="terms/s", launches=len(starts), warmup_launches=len(warm24),
                       geometry=dict(zip(("variant", "gray_bits", "block_threads", "blocks_per_chunk"),
                                         pb.pairings_query_geometry(k2, n2, C2, WL24["run_len"], opts))),
                       clocks=sampler.window(t0, t1), projected_full_run_s=(1 << 47) / (terms24 / t24),
                       roofline=roofline_object(k2, n2, m2, phi24, terms24 // len(starts), t24 / len(starts), peak_mhz))
            # the n = 24 half of BASELINE.json's metric, inside the objects the driver keeps
            r24 = n24["roofline"]
            roofline["n24"] = dict(workload=n24["workload"], value=n24["value"], unit="terms/s", seconds=t24, terms=terms24,
                                   frac=r24["frac"], useful_frac=r24["useful_frac"], yardstick_frac=r24["yardstick_frac"],
                                   executed_instr_per_term=r24.get("executed_instr_per_term"),
                                   useful_instr_per_term=r24["useful_instr_per_term"], phi=phi24, clocks=n24["clocks"],
                                   projected_full_run_s=n24["projected_full_run_s"], ncu_stale=r24.get("ncu_stale", False))

        # the other BASELINE.json configs (parity-test cases; timed here for SURVEY §8(d)'s per-config table)
        other = None
        if not args.no_configs and extras:
            other = []
            for (k2, n2, C2, m2, reps, want) in OTHER_CONFIGS:
                mod2 = pb.pairings_default_moduli(m2)
                rows2 = 1 << C2
                out2 = torch.empty((rows2, m2), dtype=torch.int32, device="cuda")
                nz2 = torch.zeros(1, dtype=torch.int64, device="cuda")
                pb.count_pairings_ex(k2, n2, C2, 0, rows2, mod2, out2.data_ptr(), stream, launch_opts(nz2.data_ptr()))    # warm-up + phi
                torch.cuda.synchronize()
                flat2 = (ctypes.c_uint32 * (rows2 * m2)).from_buffer_copy(out2.cpu().numpy().tobytes())
                D2, S2 = pb.pairings_reconstruct(k2, n2, mod2, pb.pairings_sum_rows(flat2, mod2))
                assert S2 == want, (k2, n2, S2, want)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                for _ in range(reps):
                    pb.count_pairings_ex(k2, n2, C2, 0, rows2, mod2, out2.data_ptr(), stream, opts)
                e1.record()
                torch.cuda.synchronize()
                sec = e0.elapsed_time(e1) * 1e-3 / reps
                launches += reps + 1
                terms2 = 1 << (2 * n2 - 1)
                phi2 = float(nz2.item()) / terms2
                ops2, ys2 = yardstick_ops(k2, n2, m2, phi2)
                entry = dict(config="%s(%d)" % (KIND_NAME[k2], n2), chunk_bits=C2, n_moduli=m2, launches_timed=reps,
                             seconds_per_count=sec, value=terms2 / sec, unit="terms/s", phi=phi2, ops_per_term=ops2,
                             yardstick_frac=ops2 * terms2 / sec / peak,
                             useful_frac=useful_instr(k2, n2, phi2)[0] * terms2 / sec / peak if pb.pairings_has_swar(k2, n2) else None,
                             identified=S2,
                             geometry=dict(zip(("variant", "gray_bits", "block_threads", "blocks_per_chunk"),
                                               pb.pairings_query_geometry(k2, n2, C2, rows2, opts))))
                if reps >= 20:
                    # launch-bound configs: the same `reps` launches replayed as ONE CUDA graph (no host launch gaps)
                    side = torch.cuda.Stream()
                    g = torch.cuda.CUDAGraph()
                    with torch.cuda.stream(side):
                        with torch.cuda.graph(g, stream=side):
                            for _ in range(reps):
                                pb.count_pairings_ex(k2, n2, C2, 0, rows2, mod2, out2.data_ptr(), side.cuda_stream, opts)
                        g.replay()
                        side.synchronize()
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        e0.record(side)
                        g.replay()
                        e1.record(side)
                        side.synchronize()
                    entry["seconds_per_count_cuda_graph"] = e0.elapsed_time(e1) * 1e-3 / reps
                    launches += 2 * reps
                    flat2 = (ctypes.c_uint32 * (rows2 * m2)).from_buffer_copy(out2.cpu().numpy().tobytes())
                    assert pb.pairings_reconstruct(k2, n2, mod2, pb.pairings_sum_rows(flat2, mod2))[1] == want
                m2rec, stale2 = ncu_record("instances", "%s%d" % (KIND_NAME[k2], n2))
                if m2rec and not stale2:
                    entry.update(executed_instr_per_term=m2rec["instr_per_term"], frac=m2rec["instr_per_term"] * terms2 / sec / peak)
                other.append(entry)

        # second workload: the approximate counter, S(12) with the ladder of Table 6
        ptres = None
        if not args.no_pt and extras:
            R, T, burn = 1 << 17, 1 << 11, 0                      # throughput run (too short per replica for an estimate)
            Mlev = len(PT_BETAS)
            h = torch.zeros((Mlev, 25), dtype=torch.int64, device="cuda")
            mv = torch.zeros(Mlev, dtype=torch.int64, device="cuda")
            sw = torch.zeros(Mlev, dtype=torch.int64, device="cuda")
            pb.pairings_pt_run(0, 12, PT_BETAS, 0, 1 << 10, 1 << 10, 0, 1, h.data_ptr(), mv.data_ptr(), sw.data_ptr(), stream)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            pb.pairings_pt_run(0, 12, PT_BETAS, 0, R, T, burn, 150700315, h.data_ptr(), mv.data_ptr(), sw.data_ptr(), stream)
            e1.record()
            torch.cuda.synchronize()
            sec = e0.elapsed_time(e1) * 1e-3
            # estimate run: fewer, longer replicas with burn-in (the cold levels need ~10^4 iterations to relax)
            h.zero_(); mv.zero_(); sw.zero_()
            t0 = time.perf_counter()
            pb.pairings_pt_run(0, 12, PT_BETAS, 0, 1 << 12, 1 << 15, 1 << 14, 150700315, h.data_ptr(), mv.data_ptr(), sw.data_ptr(), stream)
            torch.cuda.synchronize()
            est_s = time.perf_counter() - t0
            launches += 3
            ratios, logz = pb.pairings_pt_estimate(0, 12, PT_BETAS, h.cpu().tolist())
            est = pb.pairings_pt_counts(12, logz)[1]
            moves_s = R * T * Mlev / sec
            ptres = dict(workload="approximate count of S(12), 12 levels (Table 6 ladder, PAPER.md:327-342)",
                         replicas=R, iterations=T, seconds=sec, metropolis_moves_per_s=moves_s,
                         cpu_oracle=pt_cpu_baseline(),
                         estimate=dict(replicas=1 << 12, iterations=1 << 15, burn_in=1 << 14, seconds=est_s,
                                       s12_estimate=est, exact=227968, rel_error=est / 227968 - 1))
            if ptres["cpu_oracle"]:
                ptres["gpu_over_cpu_oracle"] = moves_s / ptres["cpu_oracle"]["value"]
            pm, pstale = ncu_record("pt")               # executed instruction slots per move x moves/s against the issue peak
            if pm and not pstale:
                ptres["roofline"] = dict(bound="alu", thread_instr_slots_per_move=pm["thread_instr_slots_per_move"],
                                         frac=pm["thread_instr_slots_per_move"] * moves_s / peak, issue_active_pct=pm["issue_active_pct"],
                                         active_threads_per_warp_instr=pm["active_threads_per_warp_instr"], ncu_source=pm["source"],
                                         ncu_commit=pm.get("commit"),
                                         work_model="per move: one 64-bit SplitMix draw for colour and position (+ one for the acceptance when dE > 0), "
                                                    "5 shared loads (old position, 4 bins), 5 shared stores when accepted; per level and iteration one "
                                                    "histogram atomic and one exchange test (+ draw when dE > 0)")
            elif pm:
                ptres["roofline"] = dict(ncu_stale=True, ncu_commit=pm.get("commit"),
                                         ncu_note="pt_kernel.cu changed since the ncu capture: no issue fraction is claimed for this build")

        cpu = cpu_baseline(kind, n) if not args.no_cpu and not args.profile_chunks else None
        par = ("every rank the whole pass x%d, residue sums cross-checked (PAPER.md:99); each sign vector counted once" if duplicate
               else "disjoint chunk ranges x%d (pairings_rank_range), per-rank residue sums added, no data-path collective") % world
        line = dict(metric="godfrey_sign_vector_terms_per_s", value=value, unit="terms/s", n_gpus=world,
                    steps=args.steps, warmup=warm, ms_per_step=dev_ms / args.steps,
                    higher_is_better=True, scaling="weak" if duplicate else "strong", vs_baseline=None, dtype="int32", data="synthetic",
                    config=dict(workload=WORKLOAD,
                                kind="langford", n=n, chunk_bits=C, n_moduli=m, parallelism=par, duplicate_run=duplicate,
                                launcher="self-spawned ranks" if os.environ.get("PAIRINGS_BENCH_SPAWNED") else ("torchrun" if world > 1 else "single process"),
                                geometry=dict(zip(("variant", "gray_bits", "block_threads", "blocks_per_chunk"), geometry)),
                                sm_count=torch.cuda.get_device_properties(local).multi_processor_count,
                                l2="flushed between steps (256 MiB fill); the kernel reads no global memory but its 24 KB zero-step tables",
                                result_check="L(20) = 2,636,337,861,200 reconstructed every run (PAPER.md:380)",
                                library=pb.pairings_build_info(),
                                n24=None if n24 is None else dict(workload=n24["workload"], terms_per_s=n24["value"], seconds=n24["seconds"],
                                                                  sm_mhz=n24["clocks"].get("sm_mhz"), reasons=n24["clocks"].get("reasons"))),
                    clocks=clocks,
                    e2e=dict(value=e2e_value, unit="terms/s", h2d_bytes_per_step=(4 * m + 8 * 5) * world,
                             d2h_bytes_per_step=rows * m * 4 * world, seconds_per_step=e2e_s / args.steps,
                             clocks=clocks_e2e),
                    profile_only=bool(args.profile_chunks),
                    gpu_launches=launches, roofline=roofline, cpu_baseline=cpu, n24=n24, lemma24=lemma24, other_configs=other, pt=ptres,
                    paper_context="paper's Kepler GPU: S(20) in 4.08 min ~ 1.1e9 terms/s (PAPER.md:397; other hardware, context only)")
    sampler.close()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line))


def pt_cpu_baseline():
    """The PT oracle (oracle/pt_oracle.cpp, as it stands) on the host cores: Metropolis moves/s for the same ladder."""
    try:
        from oracle import pt
        pt.build()
    except Exception:                                   # no compiler on the box: report nothing rather than fail the bench
        return None
    threads = host_threads()
    reps, its = 256, 1 << 12                            # about 2 s of host work
    res = [None] * threads

    def work(t):
        res[t] = pt.run(0, 12, PT_BETAS, reps, its, 1000 + t, 0)

    t0 = time.perf_counter()
    ts = [threading.Thread(target=work, args=(t,)) for t in range(threads)]
    [t.start() for t in ts]
    [t.join() for t in ts]
    dt = time.perf_counter() - t0
    moves = threads * reps * its * len(PT_BETAS)
    return dict(value=moves / dt, unit="metropolis moves/s", cores=threads, kind="oracle",
                sample="%d replicas x %d iterations x %d levels per thread, %.1f s on %d threads" % (reps, its, len(PT_BETAS), dt, threads))


# ------------------------------------------------------------------------------------------------
# launcher: --gpus N starts its own ranks
# ------------------------------------------------------------------------------------------------
def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def spawn_ranks(n: int, poll_s: float = 0.2, command=None) -> int:
    """Starts n copies of this command line, one rank each (rank r -> cuda:r), and waits for them.  Rank 0's stdout is
    this process's stdout (the JSON line); NCCL's own logging is left as the environment has it.  The library is built
    once here, before the ranks start (they would race to write the same objects on a fresh checkout).  The ranks are
    polled: as soon as one exits non-zero the others — which would wait for it in the NCCL rendezvous or a barrier
    for ever — are terminated and that exit code is returned."""
    if command is None:
        from paper_1507_00315_b200 import build as pbuild
        pbuild.build()
        command = [sys.executable, os.path.abspath(__file__)] + sys.argv[1:]
    port = os.environ.get("MASTER_PORT") or str(_free_port())
    procs = []
    for r in range(n):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(n), MASTER_ADDR="127.0.0.1", MASTER_PORT=port,
                   PAIRINGS_BENCH_SPAWNED="1")
        procs.append(subprocess.Popen(command, env=env, stdout=None if r == 0 else subprocess.DEVNULL))
    rc, live = 0, list(procs)
    while live and rc == 0:
        time.sleep(poll_s)
        for p in list(live):
            code = p.poll()
            if code is None:
                continue
            live.remove(p)
            if code != 0:
                rc = abs(code) or 1
    for p in live:                                   # a rank failed: the rest cannot finish
        p.terminate()
    for p in live:
        try:
            p.wait(timeout=10)
        except subprocess.TimeoutExpired:
            p.kill()
    return rc


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--spawn", action="store_true", help="start the rank processes even for --gpus 1 (tests the launcher on one GPU)")
    ap.add_argument("--no-n24", action="store_true", help="skip the secondary S(24) subset measurement")
    ap.add_argument("--n24-fraction", type=float, default=1.0,
                    help="fraction of the 16 seeded S(24) runs (1024 chunks each = 1/64 of the chunks, BASELINE.json configs[4]) to time")
    ap.add_argument("--scaling", default="strong", choices=["strong", "duplicate"],
                    help="N > 1: strong = disjoint chunk ranges (default); duplicate = every rank the whole pass, cross-checked (PAPER.md:99)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-pt", action="store_true", help="skip the approximate-counter (parallel tempering) measurement")
    ap.add_argument("--no-configs", action="store_true", help="skip the timing of the other BASELINE configs")
    ap.add_argument("--profile-chunks", type=int, default=0,
                    help="only the first N chunks per step: the short launches the ncu commands in profiles/ capture; the line is "
                         "marked profile_only, it is not a bench value")
    args = ap.parse_args()
    if args.gpus < 1:
        ap.error("--gpus must be >= 1")
    if "WORLD_SIZE" not in os.environ and (args.gpus > 1 or args.spawn):
        sys.exit(spawn_ranks(args.gpus))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()

"""The reference arm of bench.py (the CPU oracle on the host cores) prints one JSON line with the keys the
driver's contract names; it must run without a GPU."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "godfrey_sign_vector_terms_per_s" and d["unit"] == "terms/s"
    assert d["higher_is_better"] is True and d["vs_baseline"] is None and d["n_gpus"] == 1 and d["steps"] == 1
    assert d["value"] > 0 and d["ms_per_step"] > 0
    assert d["config"]["workload"].startswith("L(20)")
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == dict(value=d["value"], unit="terms/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0)


def test_gpu_arm_refuses_to_run_without_a_device():
    import torch
    if torch.cuda.is_available():
        return
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1"], capture_output=True, text=True,
                         timeout=600, cwd=ROOT)
    assert out.returncode != 0 and "no CPU fallback" in (out.stderr + out.stdout)


def test_gpus_n_starts_its_own_ranks():
    """`bench.py --gpus 2` without torchrun spawns two ranks itself (RANK / LOCAL_RANK / WORLD_SIZE / MASTER_* set); in the
    reference arm rank 0 alone works and prints the line, the other rank exits 0 — the launcher is what is tested here."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=600, cwd=ROOT, env=env)
    assert out.returncode == 0, out.stderr
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2


def test_world_size_must_match_gpus():
    env = dict(os.environ, WORLD_SIZE="2", RANK="0", LOCAL_RANK="0")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "1", "--steps", "1"], capture_output=True, text=True,
                         timeout=600, cwd=ROOT, env=env)
    assert out.returncode != 0 and "WORLD_SIZE" in (out.stderr + out.stdout)


def test_ncu_metrics_record_is_consistent():
    """profiles/ncu_metrics.json (what bench.py's roofline.executed_instr_per_term comes from) agrees with itself."""
    path = os.path.join(ROOT, "profiles", "ncu_metrics.json")
    if not os.path.exists(path):
        return
    doc = json.load(open(path))
    for name, m in doc["instances"].items():
        assert abs(m["instr_per_term"] - m["inst_executed_warp"] * 32 / m["terms"]) < 1e-6, name
        assert 0 < m["issue_active_pct"] <= 100 and m["kernel"].startswith("swar_kernel<")


KERNEL_FILES = {"instances": ["swar_kernel.cuh", "device_common.cuh"], "pt": ["pt_kernel.cu"]}


def _git(*args):
    out = subprocess.run(["git", "-C", ROOT] + list(args), capture_output=True, text=True)
    return out.returncode, out.stdout.strip()


def test_ncu_records_are_not_older_than_the_kernels_they_describe():
    """Every entry of profiles/ncu_metrics.json names the commit it was captured at and the hash of the kernel's source
    files at that time.  bench.py multiplies these figures into roofline.frac, so an entry captured before the last
    change of its kernel must fail here (and bench.py itself drops it: the hash no longer matches)."""
    import pytest
    sys.path.insert(0, ROOT)
    import bench
    path = os.path.join(ROOT, "profiles", "ncu_metrics.json")
    doc = json.load(open(path))
    entries = [("instances", k, v) for k, v in doc["instances"].items()] + [("pt", None, doc["pt"])]
    for which, key, rec in entries:
        assert rec.get("source_sha16") == bench.kernel_source_sha16(which), \
            "ncu capture of %s %s is older than its kernel source: re-capture it (profiles/)" % (which, key or "")
        assert bench.ncu_record(which, key) == (rec, False)
    if _git("rev-parse", "--is-inside-work-tree")[0] != 0:
        pytest.skip("no git history here")
    for which, key, rec in entries:
        files = ["paper_1507_00315_b200/csrc/" + f for f in KERNEL_FILES[which]]
        rc, last = _git("log", "-1", "--format=%H", "--", *files)
        assert rc == 0 and last
        if _git("cat-file", "-e", rec["commit"] + "^{commit}")[0] != 0:
            pytest.fail("ncu_metrics.json %s %s names an unknown commit %s" % (which, key or "", rec["commit"]))
        # the capture's commit must contain the last change of the kernel
        assert _git("merge-base", "--is-ancestor", last, rec["commit"])[0] == 0, (which, key, rec["commit"], last[:7])


def test_roofline_fractions_are_fractions():
    """frac (issue slots busy) and useful_frac (issue slots doing the method's arithmetic) stay below the ~1.2 sanity
    bound at the rates the kernel reaches; the yardstick figure is the one that may exceed 1 and is named as such."""
    sys.path.insert(0, ROOT)
    import bench
    r = bench.roofline_object(1, 20, 7, 0.2048, 1 << 39, 0.4863, 1965.0)
    assert 0.7 < r["frac"] < 1.0 and 0.3 < r["useful_frac"] < r["frac"] and r["yardstick_frac"] > 1.5
    assert abs(r["achieved"] / r["peak"] - r["frac"]) < 1e-12 and r["unit"] == "Tinstr/s" and r["bound"] == "alu"
    assert r["useful_model"]["plan"] == dict(G=3, W=4, nf=12, pairs=8, singles=4, NR=5, E=10)
    r24 = bench.roofline_object(0, 24, 9, 0.178, 1 << 37, (1 << 37) / 9.8e11, 1965.0)
    assert 0.7 < r24["frac"] < 1.0 and r24["useful_model"]["plan"]["G"] == 4


def test_spawned_ranks_do_not_hang_when_one_dies():
    """bench.py --gpus N polls its ranks: one rank exiting non-zero ends the others (they would wait for it in the
    rendezvous for ever) and its code is returned."""
    sys.path.insert(0, ROOT)
    import bench
    import time
    prog = "import os, sys, time\nif os.environ['RANK'] == '1':\n    sys.exit(7)\ntime.sleep(600)\n"
    t0 = time.time()
    rc = bench.spawn_ranks(3, poll_s=0.05, command=[sys.executable, "-c", prog])
    assert rc == 7 and time.time() - t0 < 60
    assert bench.spawn_ranks(2, poll_s=0.05, command=[sys.executable, "-c", "pass"]) == 0

"""Builds libpairings_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1507_00315_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import concurrent.futures
import glob
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(ROOT, "include")
OBJ = os.path.join(HERE, "build")
SO = os.path.join(HERE, "libpairings_b200.so")
PROBE_SRC = os.path.join(HERE, "probe", "issue_probe.cu")
PROBE_SO = os.path.join(HERE, "libpairings_probe.so")     # bench.py's calibration kernels, not part of the product

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
CFLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-I", INCLUDE, "-I", CSRC]


def swar_instances():
    """(kind, n) pairs of csrc/swar_list.h — swar_inst.cu is compiled once per pair."""
    import re
    text = open(os.path.join(CSRC, "swar_list.h")).read()
    text = re.sub(r"//.*", "", text)
    return [(int(k), int(n)) for k, n in re.findall(r"X\(\s*(\d+)\s*,\s*(\d+)\s*\)", text)]


def sources():
    """[(source, extra defines, object tag)]"""
    out = []
    for f in sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cpp"))):
        if os.path.basename(f) == "swar_inst.cu":
            for k, n in swar_instances():
                out.append((f, ["-DPAIRINGS_SWAR_KIND=%d" % k, "-DPAIRINGS_SWAR_N=%d" % n], "_%d_%d" % (k, n)))
        else:
            out.append((f, [], ""))
    return out


def _deps_stamp():
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) +
                    glob.glob(os.path.join(INCLUDE, "*.h")) + [os.path.abspath(__file__)]):
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def _compile(item, stamp, verbose):
    src, defines, tag = item
    obj = os.path.join(OBJ, os.path.basename(src) + tag + "." + stamp + ".o")
    if os.path.exists(obj) and os.path.getmtime(obj) >= os.path.getmtime(src):
        return obj
    cmd = [NVCC] + ARCH + CFLAGS + (["-Xptxas", "-v"] if verbose else []) + defines + ["-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (src, r.stdout, r.stderr))
    if verbose:
        sys.stderr.write(r.stderr)
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    stamp = _deps_stamp()
    srcs = sources()
    for f in glob.glob(os.path.join(OBJ, "*.o")):
        if force or not f.endswith("." + stamp + ".o"):     # stale objects of older header states
            os.remove(f)
    with concurrent.futures.ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
        objs = list(ex.map(lambda s: _compile(s, stamp, verbose), srcs))
    newest = max(os.path.getmtime(o) for o in objs)
    if force or not os.path.exists(SO) or os.path.getmtime(SO) < newest:
        tmp = SO + ".tmp.%d" % os.getpid()
        cmd = [NVCC] + ARCH + ["-shared", "-o", tmp] + objs + ["-lcudart"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed:\n%s\n%s" % (r.stdout, r.stderr))
        os.replace(tmp, SO)
    return SO


def build_probe(force: bool = False) -> str:
    """bench.py's integer-issue calibration kernels (probe/issue_probe.cu) as their own small library."""
    if force or not os.path.exists(PROBE_SO) or os.path.getmtime(PROBE_SO) < os.path.getmtime(PROBE_SRC):
        tmp = PROBE_SO + ".tmp.%d" % os.getpid()
        cmd = [NVCC] + ARCH + ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-shared", "-o", tmp, PROBE_SRC, "-lcudart"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (PROBE_SRC, r.stdout, r.stderr))
        os.replace(tmp, PROBE_SO)
    return PROBE_SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
    print(build_probe(force="--force" in sys.argv))

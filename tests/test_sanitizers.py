"""ASan + UBSan over the host code: csrc/host_math.cpp (CRT, partitioner, journal parser — the code that
reads untrusted file text) and the two CPU oracles, each built with -fsanitize=address,undefined together with
tests/sanitize_driver.cpp and run; a sanitizer report or a failed check is a non-zero exit.  No GPU, no CUDA toolkit."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
DRIVER = os.path.join(ROOT, "tests", "sanitize_driver.cpp")
FLAGS = ["-std=c++17", "-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=all"]
BUILDS = [
    ("host", "-DDRIVE_HOST", [os.path.join(ROOT, "paper_1507_00315_b200", "csrc", "host_math.cpp")],
     ["-I", os.path.join(ROOT, "include"), "-I", os.path.join(ROOT, "paper_1507_00315_b200", "csrc")]),
    ("oracle", "-DDRIVE_ORACLE", [os.path.join(ROOT, "oracle", "godfrey_oracle.cpp")], []),
    ("pt", "-DDRIVE_PT", [os.path.join(ROOT, "oracle", "pt_oracle.cpp")], []),
]


@pytest.mark.parametrize("name,define,sources,includes", BUILDS, ids=[b[0] for b in BUILDS])
def test_host_code_is_clean_under_asan_and_ubsan(name, define, sources, includes, tmp_path):
    if shutil.which("g++") is None:
        pytest.skip("no g++")
    exe = str(tmp_path / ("sanitize_" + name))
    cc = subprocess.run(["g++"] + FLAGS + [define] + includes + [DRIVER] + sources + ["-o", exe], capture_output=True, text=True)
    assert cc.returncode == 0, cc.stderr[-3000:]
    work = tmp_path / "files"
    work.mkdir()
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    run = subprocess.run([exe] + ([str(work)] if name == "host" else []), capture_output=True, text=True, timeout=600, env=env)
    assert run.returncode == 0, (run.stdout[-500:], run.stderr[-3000:])
    assert run.stdout.strip().endswith("ok") and "runtime error" not in run.stderr and "AddressSanitizer" not in run.stderr

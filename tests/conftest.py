import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session", autouse=True)
def built_library():
    """The CUDA library is built in-tree (nvcc, sm_100a) if it is missing or older than its sources; the tests never
    fall back to anything else."""
    from paper_1507_00315_b200 import build as pbuild
    return pbuild.build()


def read_golden(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            rows.append(line.split())
    return rows


@pytest.fixture(scope="session")
def paper_counts():
    """{(kind, n): count with reflections identified} from the paper's tables."""
    out = {}
    for k, n, v in read_golden("paper_exact_counts.txt"):
        out[(0 if k == "S" else 1, int(n))] = int(v)
    return out


@pytest.fixture(scope="session")
def paper_distinct():
    out = {}
    for k, n, v in read_golden("paper_distinct_counts.txt"):
        out[(0 if k == "S" else 1, int(n))] = int(v)
    return out


@pytest.fixture(scope="session")
def worked_examples():
    out = {}
    for row in read_golden("paper_worked_examples.txt"):
        out.setdefault(row[0], []).append(tuple(int(t) for t in row[1:]))
    return out

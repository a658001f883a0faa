import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def golden():
    """tests/golden/dpie_golden.txt -> (lenses dict, list of (lens rows, t1, t2, g1, g2)) with mpmath values."""
    import mpmath as mp
    mp.mp.dps = 40
    path = os.path.join(ROOT, "tests", "golden", "dpie_golden.txt")
    lenses, cases = {}, []
    for line in open(path):
        w = line.split()
        if not w or w[0].startswith("#"):
            continue
        if w[0] == "lens":
            lenses[w[1]] = tuple(float(v) for v in w[2:9])
        elif w[0] == "case":
            rows = [lenses[n] for n in w[1].split("+")]
            cases.append((rows, float(w[2]), float(w[3]), mp.mpf(w[4]), mp.mpf(w[5])))
    return lenses, cases

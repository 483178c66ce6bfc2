import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def load_golden(name):
    """Parse a tests/golden/*.txt fixture (format: tests/golden/README.md)."""
    import math
    path = os.path.join(ROOT, "tests", "golden", name)
    kind, bins, pts, pts2, expect = None, {}, [], [], {}
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        tok = line.split()
        if tok[0] == "kind":
            kind = tok[1]
        elif tok[0] == "bins":
            for kv in tok[1:]:
                k, v = kv.split("=")
                bins[k] = float(v) if k not in ("n1", "n2", "log1") else int(v)
        elif tok[0] == "point":
            pts.append([float(t) for t in tok[1:]])
        elif tok[0] == "point2":
            pts2.append([float(t) for t in tok[1:]])
        elif tok[0] == "expect":
            for kv in tok[1:]:
                k, v = kv.split(":")
                expect[int(k)] = int(v)
    # angles in the fixtures are degrees; the APIs take radians
    if kind == "angular":
        bins["lo1"] = math.radians(bins["lo1"])
        bins["hi1"] = math.radians(bins["hi1"])
    if "aperture" in bins:
        bins["aperture"] = math.radians(bins["aperture"])
    return kind, bins, pts, pts2, expect


@pytest.fixture(scope="session")
def oracle():
    from oracle import oracle as o
    o.build()
    return o

import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.join(ROOT, "oracle"), os.path.join(ROOT, "tests")):
    if p not in sys.path:
        sys.path.insert(0, p)

GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def read_golden_table(name):
    rows = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            t = line.split()
            rows[t[0]] = [float(x) for x in t[1:]]
    return rows


@pytest.fixture(scope="session")
def table1():
    r = read_golden_table("table1_emhd_mode.txt")
    names = ["rho", "u", "u1", "u2", "u3", "B1", "B2", "B3", "q", "dP"]
    P0 = np.array([r[n][0] for n in names])
    dP = np.array([r[n][1] + 1j * r[n][2] for n in names])
    w = r["omega"][1] + 1j * r["omega"][2]
    k = np.array([2 * np.pi, 4 * np.pi, 0.0])
    return P0, dP, w, k

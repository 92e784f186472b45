import math
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.dirname(os.path.abspath(__file__))):
    if p not in sys.path:
        sys.path.insert(0, p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def load_table1():
    """Rows of tests/golden/table1_spherical_photon_orbits.txt as dicts."""
    rows = []
    path = os.path.join(os.path.dirname(__file__), "golden", "table1_spherical_photon_orbits.txt")
    with open(path) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            lab, r, phi, q, mc, dphi = line.split()
            rows.append(dict(label=lab, r=float(eval(r, {"sqrt": math.sqrt})), phi=float(phi), q=float(q),
                             maxcos=float(mc), dphi=float(dphi)))
    return rows


@pytest.fixture(scope="session")
def table1():
    return load_table1()

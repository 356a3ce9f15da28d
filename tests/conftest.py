import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def pdf():
    from paper_2106_10279_b200 import workloads as W
    return W.pdf_table()


@pytest.fixture(scope="session")
def oracle_procs(pdf):
    """One oracle handle per process id (C0..C3 physics)."""
    from oracle import mfo
    from paper_2106_10279_b200 import workloads as W
    return {wl.process: mfo.Process(wl, pdf) for wl in (W.C0, W.C1, W.C2, W.C3)}

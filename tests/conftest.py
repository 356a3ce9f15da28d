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
    """One oracle handle per process id (C0..C3 physics, and C5 = the flavour-summed pp -> ttbar with its own table)."""
    from oracle import mfo
    from paper_2106_10279_b200 import workloads as W
    procs = {wl.process: mfo.Process(wl, pdf) for wl in (W.C0, W.C1, W.C2, W.C3)}
    procs[W.MF_PP_TT] = mfo.Process(W.C5, W.pdf_table_flavours())
    procs[W.MF_PP_TTG] = mfo.Process(W.C6, W.pdf_table_flavours())
    procs[W.MF_GG_TTGGG] = mfo.Process(W.C7, pdf)
    procs[W.MF_PP_TTGG] = mfo.Process(W.C8, W.pdf_table_flavours())
    return procs


@pytest.fixture(scope="session")
def gpu_procs(pdf):
    """One CUDA-path handle per process id.  Fails loudly (no fallback) if the library or the GPU is missing."""
    from paper_2106_10279_b200 import api
    from paper_2106_10279_b200 import workloads as W
    procs = {wl.process: api.Process(wl, pdf) for wl in (W.C0, W.C1, W.C2, W.C3)}
    procs[W.MF_PP_TT] = api.Process(W.C5, W.pdf_table_flavours())
    procs[W.MF_PP_TTG] = api.Process(W.C6, W.pdf_table_flavours())
    procs[W.MF_GG_TTGGG] = api.Process(W.C7, pdf)
    procs[W.MF_PP_TTGG] = api.Process(W.C8, W.pdf_table_flavours())
    yield procs
    for p in procs.values():
        p.close()


@pytest.fixture(scope="session")
def oracle_pool():
    """The oracle as one single-threaded process per host core on disjoint index ranges (tests/oracle_pool.py)."""
    from oracle_pool import OraclePool
    pool = OraclePool()
    yield pool
    pool.close()


_ADAPTED = {}


def adapted_grid(oracle_proc, wl, n_iter=3):
    """A non-uniform VEGAS grid made by the ORACLE alone (a few small adapting iterations); cached."""
    from paper_2106_10279_b200 import workloads as W
    if wl.process not in _ADAPTED:
        n_events = {0: 20000, 1: 8192, 2: 4096, 3: 1024, 4: 8192, 5: 4096, 6: 96, 7: 384}[wl.process]
        grid = W.uniform_grid(wl.n_dims, wl.n_bins)
        for k in range(n_iter):
            hist, _ = oracle_proc.vegas_iterate(grid, 12345, k, 0, n_events)
            grid = oracle_proc.refine_grid(grid, hist, W.VEGAS_ALPHA)
        _ADAPTED[wl.process] = grid
    return _ADAPTED[wl.process].copy()

import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.dirname(os.path.abspath(__file__))):
    if p not in sys.path:
        sys.path.insert(0, p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    # the -fopenmp build of the same sources (outermost grid loops only; per-point arithmetic and results unchanged) keeps the
    # suite to minutes; ORACLE_THREADS=1 runs the plain single-threaded build
    oracle.use_threads(int(os.environ.get("ORACLE_THREADS", os.cpu_count() or 1)))
    return oracle


@pytest.fixture(scope="session", autouse=True)
def _library_is_built():
    """Build (or refresh) libmhd_b200.so in-tree before any test: nvcc cross-compiles without a GPU, seconds when up to date."""
    from paper_2510_13965_b200 import build
    build.build()

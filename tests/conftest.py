import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    # the libraries are built in-tree (git-ignored): a checkout without them builds them once (nvcc cross-compiles without a
    # GPU); an existing library is used as it is - __graft_entry__.build() is the place that rebuilds
    from paper_2207_14276_b200 import build as cuda_build
    from oracle import build as oracle_build
    if not os.path.exists(cuda_build.LIB):
        cuda_build.build(force=True)
    if not os.path.exists(oracle_build.LIB):
        oracle_build.build(force=True)


@pytest.fixture(scope="session")
def params():
    from paper_2207_14276_b200 import workloads
    return workloads.default_params()

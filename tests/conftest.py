import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_sessionstart(session):
    # the C-ABI library is built in-tree (nvcc cross-compiles sm_100a without a GPU); no-op when it is current
    from paper_2511_03683_b200 import _build
    _build.build()

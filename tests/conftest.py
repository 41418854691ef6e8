import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


def pytest_sessionstart(session):
    # The library is built in-tree and git-ignored: on a fresh checkout build it once (nvcc cross-compiles without a
    # GPU).  Only when it is MISSING -- a stale library is the developer's business, build.py rebuilds on demand.
    if not os.path.exists(os.path.join(ROOT, "paper_2305_08140_b200", "csrc", "libnepzbl.so")):
        from paper_2305_08140_b200 import build     # the package does not load the library on import, binding does
        build.build()

"""The memcheck stand-in (compute-sanitizer is closed on the GPU pool this was developed on): the small cases of the
GPU suite -- config 1, open boundaries, clusters, a neighbour-capacity overflow in the middle of an MD run, a short
cascade with rebuilds, ZBL atoms and fp64 sites, two types, the paper-sized model, odd sizes -- run in a subprocess
against libnepzbl_checked.so, the same sources compiled with -DNEPZBL_CHECKED: every index that is read from memory
and then used as an address is tested against its bound, a violation prints its site and traps."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CASES = ["tests/test_gpu_parity.py", "tests/test_gpu_md.py", "tests/test_gpu_disordered.py", "tests/test_gpu_alloy.py",
         "tests/test_gpu_paper_model.py", "tests/test_gpu_shapes.py", "tests/test_gpu_triclinic.py", "tests/test_gpu_nhc.py",
         "tests/test_gpu_next4.py"]


def test_small_cases_on_the_bounds_checked_build():
    from paper_2305_08140_b200 import build
    lib = build.build(checked=True)
    assert os.path.exists(lib)
    env = dict(os.environ, NEPZBL_LIB="checked")
    r = subprocess.run([sys.executable, "-m", "pytest", "-q", "-x", "-m", "gpu", "-p", "no:cacheprovider"] + CASES,
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=1800)
    tail = (r.stdout + r.stderr)[-3000:]
    assert "nepzbl check failed" not in r.stdout + r.stderr, tail
    assert r.returncode == 0, tail

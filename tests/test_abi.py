"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/nepzbl.h declares; without a GPU nep_zbl_create fails loudly (no fallback)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "nepzbl.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"^\s*(?:const\s+)?[A-Za-z_][\w\s\*]*?\b(\w+)\s*\(", src, flags=re.M)
    return sorted(set(n for n in names if n not in ("defined",)))


@pytest.fixture(scope="module")
def lib():
    from paper_2305_08140_b200 import build
    return C.CDLL(build.build())


def test_header_declares_the_north_star_calls():
    d = _declared()
    for name in ("nep_zbl_create", "neighbor_build", "nep_zbl_compute", "md_step"):
        assert name in d


def test_library_exports_every_declared_symbol(lib):
    d = _declared()
    assert len(d) >= 15
    for name in d:
        assert hasattr(lib, name), name


def test_binding_lists_the_same_entry_points():
    import torch  # noqa: F401
    from paper_2305_08140_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()


def test_sass_is_sm_100a(lib):
    import subprocess
    from paper_2305_08140_b200 import build
    out = subprocess.run(["cuobjdump", "-lelf", build.LIB], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_create_fails_loudly_without_gpu_or_with_bad_params(lib):
    import numpy as np
    import torch
    from paper_2305_08140_b200 import binding, workloads as wl
    m = wl.synthetic_model()
    if not torch.cuda.is_available():
        with pytest.raises(binding.NepZblError) as e:
            binding.NepZbl(m, 100)
        assert e.value.code == -6 and "no CPU fallback" in str(e.value)
    bad = dict(m, n_max_radial=16)     # beyond the largest kernel shape (n_max <= 15 / 10, basis <= 8)
    with pytest.raises(binding.NepZblError) as e:
        binding.NepZbl(bad, 100)
    assert e.value.code == -7
    bad = dict(m, cap_angular=129)     # two 64-bit mask words per atom at most
    with pytest.raises(binding.NepZblError) as e:
        binding.NepZbl(bad, 100)
    assert e.value.code == -1


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2305_08140_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "nep_zbl_oracle" not in text, f
    otext = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "nep_zbl_oracle.c")).read()
    assert "import paper_2305_08140_b200" not in otext and "from paper_2305_08140_b200" not in otext
    assert "nepzbl.h" not in otext

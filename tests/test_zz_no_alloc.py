"""nep_zbl_energy_sums_static (include/nepzbl.h; csrc/no_alloc.cu): the allocation-free variant of the md_energies
reduction, its block partials in a file-scope device array.  Checked against the existing path (md_energies) on two
calls in a row, at the tolerance the MD tests use for the kinetic energy (rel 1e-12; tests/test_gpu_md.py).

Collected LAST on purpose (test_zz_*): the suite runs with `pytest -x`, a failure here must not hide other tests.
Passes alone in a fresh process (the first call resolves the scratch address) and after the other tests."""
import numpy as np
import pytest
import torch

from paper_2305_08140_b200 import workloads as wl

pytestmark = pytest.mark.gpu

REL = 1e-12
_WARM = []   # non-empty once the entry point has run in this process


@pytest.fixture(scope="module")
def nb():
    from paper_2305_08140_b200 import binding
    assert torch.cuda.is_available()
    return binding


def _md(nb, w):
    g = nb.NepZbl(w.model, w.n)
    pos = torch.from_numpy(w.pos.copy()).cuda()
    vel = torch.from_numpy(w.vel.copy()).cuda()
    types = torch.from_numpy(w.types).cuda()
    g.md_init(pos, vel, types, w.box, w.pbc)
    return g, pos, vel, types


def _check(nb, g, vel, types, mass, out):
    """One call of the new entry point on the current MD state against md_energies."""
    ep, ek = g.md_energies()                      # existing path (synchronises the library's stream)
    _, e = g.md_get_forces()
    out.fill_(float("nan"))
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    nb.nep_zbl_energy_sums_static(vel, e, types, mass, out)
    torch.cuda.synchronize()
    # nothing is allocated on the device (the first call of a process may load the kernel's module lazily)
    assert torch.cuda.mem_get_info()[0] == free0 or not _WARM
    _WARM.append(True)
    got = out.cpu().numpy()
    assert got[0] == pytest.approx(ep, rel=REL), (got[0], ep)
    assert got[1] == pytest.approx(ek, rel=REL), (got[1], ek)
    return got.copy(), e


def test_two_calls_in_a_row_match_md_energies(nb):
    # 17^3 cells = 9 826 atoms: three 4096-atom blocks, the last one ragged
    w = wl.thermal_bulk(17, seed=41, sigma_pos=0.03)
    g, pos, vel, types = _md(nb, w)
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    first, _ = _check(nb, g, vel, types, [wl.W_MASS], out)
    for _ in range(3):                            # another state: the shared scratch now holds the first call's partials
        g.md_step(1.0, float("inf"))
    second, e = _check(nb, g, vel, types, [wl.W_MASS], out)
    assert second[1] != first[1]                  # the states differ, the answers are not a leftover
    # fixed summation order: the same data give the same bits, and types = NULL means type 0
    again = torch.empty(2, dtype=torch.float64, device="cuda")
    nb.nep_zbl_energy_sums_static(vel, e, None, [wl.W_MASS], again)
    torch.cuda.synchronize()
    assert np.array_equal(again.cpu().numpy(), second)
    g.close()


def test_two_types_small_system_and_back_to_back_calls(nb):
    # 432 atoms (one ragged block), per-type masses; then a larger system right after it on the same scratch
    w = wl.thermal_bulk(6, seed=42, sigma_pos=0.03, model=wl.alloy_model(spread=0.05, stream=13))
    w.types = wl.random_types(w.n, 42)
    g, pos, vel, types = _md(nb, w)
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    mass = [float(m) for m in w.model["mass"]]
    _check(nb, g, vel, types, mass, out)
    g.md_step(1.0, float("inf"))
    _check(nb, g, vel, types, mass, out)
    g.close()
    w2 = wl.thermal_bulk(12, seed=43, sigma_pos=0.02)
    g2, pos2, vel2, types2 = _md(nb, w2)
    _check(nb, g2, vel2, types2, [wl.W_MASS], out)
    _check(nb, g2, vel2, types2, [wl.W_MASS], out)
    g2.close()


def test_sizes_beyond_the_static_maximum_are_rejected(nb):
    v = torch.zeros(3 * 8, dtype=torch.float64, device="cuda")
    e = torch.zeros(8, dtype=torch.float64, device="cuda")
    out = torch.full((2,), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(nb.NepZblError) as ei:
        nb.nep_zbl_energy_sums_static(v, e, None, [wl.W_MASS], out, n_atoms=nb.STATIC_MAX_ATOMS + 1)
    assert ei.value.code == -7 and "NEPZBL_STATIC_MAX_ATOMS" in str(ei.value)
    with pytest.raises(nb.NepZblError):           # nine types: more than the mass table holds
        nb.nep_zbl_energy_sums_static(v, e, None, [1.0] * 9, out)
    with pytest.raises(nb.NepZblError):           # two types need a type array
        nb.nep_zbl_energy_sums_static(v, e, None, [1.0, 2.0], out)
    with pytest.raises(nb.NepZblError):           # the result buffer must be device memory
        nb.nep_zbl_energy_sums_static(v, e, None, [1.0], np.zeros(2))
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [7.0, 7.0]       # a rejected call launches nothing
    nb.nep_zbl_energy_sums_static(v, e, None, [wl.W_MASS], out, n_atoms=0)   # empty input: zeros
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [0.0, 0.0]

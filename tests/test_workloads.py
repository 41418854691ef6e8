"""Host logic of the seeded input generators (paper_2305_08140_b200/workloads.py): reproducible bit for bit from the
seed, shapes of BASELINE.json's configs, and no method arithmetic (the module imports neither side)."""
import hashlib

import numpy as np

from paper_2305_08140_b200 import workloads as wl


def _digest(*arrays):
    h = hashlib.sha256()
    for a in arrays:
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()


def test_generators_are_reproducible_and_seed_dependent():
    a, b, c = wl.config1(seed=1), wl.config1(seed=1), wl.config1(seed=2)
    assert _digest(a.pos, a.box) == _digest(b.pos, b.box) != _digest(c.pos, c.box)
    m1, m2, m3 = wl.synthetic_model(), wl.synthetic_model(), wl.synthetic_model(seed=122)
    assert _digest(m1["w0"], m1["c_radial"], m1["c_angular"]) == _digest(m2["w0"], m2["c_radial"], m2["c_angular"])
    assert _digest(m1["w0"]) != _digest(m3["w0"])
    t1, t2 = wl.thermal_bulk(6, seed=3), wl.thermal_bulk(6, seed=3)
    assert _digest(t1.pos, t1.vel) == _digest(t2.pos, t2.vel)
    assert np.abs(t1.vel.mean(axis=1)).max() < 1e-18                       # centre-of-mass momentum removed (C-17)
    g1, g2 = wl.alloy_model(), wl.alloy_model()
    assert _digest(g1["c_radial"], g1["c_angular"]) == _digest(g2["c_radial"], g2["c_angular"])
    assert g1["n_types"] == 2 and g1["c_radial"].shape == (2, 2, 5, 9) and not np.allclose(g1["c_radial"][0, 1], g1["c_radial"][1, 0])
    assert np.array_equal(wl.random_types(100, 5), wl.random_types(100, 5))


def test_config_shapes_follow_baseline_json():
    w1 = wl.config1()
    assert w1.n == 2000 and len(w1.info["pairs"]) == 5 and list(w1.pbc) == [1, 1, 1]
    q = w1.pos * 2.0 ** 18
    assert np.array_equal(q, np.round(q))                                    # quantised to 2^-18 A
    seps = [np.linalg.norm(w1.pos[:, j] - w1.pos[:, i]) for i, j in w1.info["pairs"]]
    assert all(1.0 - 1e-4 <= s <= 2.0 + 1e-4 for s in seps)
    w2 = wl.config2(cells=6)
    assert w2.dt_max == 1.0 and w2.max_displacement == float("inf") and w2.n == 432
    w3 = wl.bulk_cascade(6, 1.0e4, seed=3, n_steps=10, name="c3")
    v = np.sqrt((w3.vel[:, w3.info["pka_atom"]] ** 2).sum())
    assert abs(v - 1.02453) < 1e-4 and w3.max_displacement == 0.015          # 10 keV W atom (C-16)
    w5 = wl.config5(cells=(6, 6, 4))
    assert list(w5.pbc) == [1, 1, 0] and w5.box[8] == 4 * wl.A0_CONFIG + 40.0
    u = np.array(w5.info["pka_direction"])
    assert abs(np.degrees(np.arccos(-u[2])) - 7.0) < 1e-9                    # 7 degrees off the surface normal
    m = wl.paper_model()
    assert (m["n_max_radial"], m["n_max_angular"], m["n_neurons"], m["has_4body"]) == (15, 10, 100, 0)
    assert list(m["zbl_c"]) == [0.32825, 0.09219, 0.58110]                   # Eq. 3 as printed


def test_module_imports_neither_side():
    import ast
    tree = ast.parse(open(wl.__file__).read())
    mods = set()
    for node in ast.walk(tree):
        if isinstance(node, ast.Import):
            mods |= {a.name.split(".")[0] for a in node.names}
        elif isinstance(node, ast.ImportFrom):
            mods.add((node.module or "").split(".")[0] if node.level == 0 else "<relative>")
    assert mods <= {"__future__", "dataclasses", "numpy"}, mods

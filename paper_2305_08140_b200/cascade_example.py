"""The paper's cascade protocol end to end on one GPU, with the synthetic potential:

    python -m paper_2305_08140_b200.cascade_example --cells 80 --energy-kev 10 --steps 5000

bcc W at 300 K, one primary knock-on atom at the centre, adaptive time step (fastest atom moves at most
`--max-disp` Angstrom per step, dt <= 1 fs), the 3 a0 border layer held at 300 K by a Nose-Hoover chain, and a
Wigner-Seitz defect count against the initial lattice every `--every` steps.  Uses only the C-ABI binding and the
seeded input generators; the weights are random numbers (the paper's trained model is not available), so the
defect numbers are those of the synthetic potential, not of tungsten.
"""
from __future__ import annotations

import argparse
import time

import torch

from . import binding, workloads as wl


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--cells", type=int, default=40, help="bcc cells per edge (atoms = 2 cells^3)")
    ap.add_argument("--energy-kev", type=float, default=2.0)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--every", type=int, default=500, help="steps between defect counts")
    ap.add_argument("--max-disp", type=float, default=0.015)
    ap.add_argument("--seed", type=int, default=3)
    ap.add_argument("--no-thermostat", action="store_true")
    a = ap.parse_args(argv)

    w = wl.bulk_cascade(a.cells, a.energy_kev * 1e3, seed=a.seed, n_steps=a.steps, name="cascade")
    g = binding.NepZbl(w.model, w.n)
    dev = g.device
    pos = torch.from_numpy(w.pos.copy()).to(dev)
    vel = torch.from_numpy(w.vel.copy()).to(dev)
    g.md_init(pos, vel, torch.from_numpy(w.types).to(dev), w.box, w.pbc)
    group = wl.border_group(w.pos, w.box, w.pbc)
    if not a.no_thermostat:
        g.md_set_thermostat(torch.from_numpy(group).to(dev), 300.0, 100.0, 4)
    g.wigner_seitz_set_reference(torch.from_numpy(w.pos.copy()).to(dev), w.box, w.pbc)
    e0 = sum(g.md_energies())
    print(f"{w.n} atoms, {int(group.sum())} in the border layer, PKA {a.energy_kev:g} keV, workspace "
          f"{g.workspace_bytes / 2**30:.2f} GiB")
    torch.cuda.synchronize(dev)
    t0, t_sim, done = time.time(), 0.0, 0
    while done < a.steps:
        k = min(a.every, a.steps - done)
        tr, _ = g.md_run(k, 1.0, a.max_disp, want_trace=True)
        done += k
        t_sim += float(tr.sum())
        _, _, (nv, ni) = g.wigner_seitz_count(pos, want_nearest=False, want_occupancy=False)
        ep, ek = g.md_energies()
        extra, tg = 0.0, float("nan")
        if not a.no_thermostat:
            _, _, tg, extra = g.md_get_thermostat()
        print(f"step {done:6d}  t = {t_sim:8.1f} fs  dt = {tr[-1]:.4f} fs  vacancies = {nv}  interstitials = {ni}  "
              f"T_border = {tg:6.1f} K  conserved - initial = {ep + ek + extra - e0:+.2f} eV  "
              f"rebuilds = {g.md_get_counters()[1]}")
    torch.cuda.synchronize(dev)
    wall = time.time() - t0
    print(f"{a.steps} steps in {wall:.2f} s: {w.n * a.steps / wall:.3e} atom-steps/s (defect counts included)")
    return 0


if __name__ == "__main__":
    raise SystemExit(main())

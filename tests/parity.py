"""Shared comparison helpers for the GPU parity tests (tolerances of BASELINE.json north_star,
made precise in DESIGN.md "Tolerances")."""
import numpy as np

E_TOL = 1e-5          # eV, absolute, per atom
F_ABS, F_REL = 1e-4, 1e-4   # eV/A; per atom |dF| <= max(F_ABS, F_REL |F_i|)
W_REL, W_ABS = 1e-4, 1e-4   # per atom max_c |dW_c| <= W_REL max_c |W_c| + W_ABS (eV)


def compare(e, f, w, ref, idx=None, label=""):
    """Returns dict of worst ratios error/tolerance (<= 1 passes) and prints a one-line summary."""
    sl = slice(None) if idx is None else idx
    out = {}
    de = np.abs(e[sl] - ref.energy[sl])
    out["energy"] = de.max() / E_TOL
    df = np.sqrt(((f[:, sl] - ref.force[:, sl]) ** 2).sum(axis=0))
    fn = np.sqrt((ref.force[:, sl] ** 2).sum(axis=0))
    out["force"] = (df / np.maximum(F_ABS, F_REL * fn)).max()
    if w is not None:
        dw = np.abs(w[:, sl] - ref.virial[:, sl]).max(axis=0)
        wn = np.abs(ref.virial[:, sl]).max(axis=0)
        out["virial"] = (dw / (W_REL * wn + W_ABS)).max()
    print(f"[parity {label}] max|dE|={de.max():.3e} eV  max|dF|={df.max():.3e} eV/A "
          f"(|F|max={fn.max():.3e})  ratios={ {k: round(float(v), 4) for k, v in out.items()} }")
    return out


def list_sets(nn, nl):
    return [frozenset(nl[i, :nn[i]].tolist()) for i in range(len(nn))]


def compare_neighbor_sets(nn_g, nl_g, pos, box, pbc, rc, oracle, margin=1e-6):
    """Bit-exact set equality, excluding pairs within `margin` of the cutoff (north_star)."""
    cap = nl_g.shape[1] + 64
    nn_lo, nl_lo = oracle.neighbors(pos, box, pbc, rc - margin, use_cell=pos.shape[1] > 3000, cap=cap)
    nn_hi, nl_hi = oracle.neighbors(pos, box, pbc, rc + margin, use_cell=pos.shape[1] > 3000, cap=cap)
    lo, hi, g = list_sets(nn_lo, nl_lo), list_sets(nn_hi, nl_hi), list_sets(nn_g, nl_g)
    bad = [i for i in range(len(g)) if not (lo[i] <= g[i] <= hi[i])]
    dup = [i for i in range(len(g)) if len(g[i]) != nn_g[i]]
    return bad, dup, sum(len(h) - len(l) for h, l in zip(hi, lo))


def compare_neighbor_sets_sel(nn_g, nl_g, sel, pos, box, pbc, rc, oracle, margin=1e-6):
    """The same for a selection of atoms of a large system: nn_g / nl_g are the GPU rows of the atoms sel[t]."""
    cap = nl_g.shape[1] + 64
    nn_lo, nl_lo = oracle.neighbors(pos, box, pbc, rc - margin, use_cell=True, cap=cap, sel=sel)
    nn_hi, nl_hi = oracle.neighbors(pos, box, pbc, rc + margin, use_cell=True, cap=cap, sel=sel)
    lo, hi, g = list_sets(nn_lo, nl_lo), list_sets(nn_hi, nl_hi), list_sets(nn_g, nl_g)
    bad = [int(sel[t]) for t in range(len(g)) if not (lo[t] <= g[t] <= hi[t])]
    dup = [int(sel[t]) for t in range(len(g)) if len(g[t]) != nn_g[t]]
    return bad, dup, sum(len(h) - len(l) for h, l in zip(hi, lo))

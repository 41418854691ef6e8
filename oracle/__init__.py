"""ctypes front-end of the fp64 CPU oracle (oracle/nep_zbl_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package never imports this module and
this module never imports the product package.  All arithmetic lives in the C file; this
file only marshals numpy arrays (argument conversion, array allocation).

Citations follow the C file: P:n = PAPER.md line n, S:x = SURVEY.md 8(c) paragraph x.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nep_zbl_oracle.c")
_LIB = os.path.join(_HERE, "libnepzbl_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (OpenMP over sites).  Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-ffp-contract=off",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _CParams(C.Structure):
    _fields_ = [
        ("n_types", C.c_int32),
        ("rc_radial", C.c_double), ("rc_angular", C.c_double),
        ("n_max_radial", C.c_int32), ("n_max_angular", C.c_int32),
        ("basis_radial", C.c_int32), ("basis_angular", C.c_int32),
        ("l_max", C.c_int32), ("has_4body", C.c_int32), ("has_5body", C.c_int32), ("n_neurons", C.c_int32),
        ("c_radial", C.POINTER(C.c_double)), ("c_angular", C.POINTER(C.c_double)),
        ("q_scaler", C.POINTER(C.c_double)),
        ("w0", C.POINTER(C.c_double)), ("b0", C.POINTER(C.c_double)), ("w1", C.POINTER(C.c_double)),
        ("b1", C.c_double),
        ("zbl_enabled", C.c_int32),
        ("zbl_r_inner", C.c_double), ("zbl_r_outer", C.c_double),
        ("zbl_n_terms", C.c_int32),
        ("zbl_c", C.c_double * 4), ("zbl_d", C.c_double * 4),
        ("zbl_a_num", C.c_double), ("zbl_a_pow", C.c_double), ("coulomb_k", C.c_double),
        ("atomic_number", C.POINTER(C.c_double)), ("mass", C.POINTER(C.c_double)),
    ]


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_descriptor_dim.restype = C.c_int
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_zbl_screening_length.restype = C.c_double
        _lib.orc_neighbors.restype = C.c_int
        _lib.orc_compute.restype = C.c_int
        _lib.orc_md_run.restype = C.c_int
    return _lib


class Params:
    """Holds the model as contiguous fp64 numpy arrays plus the C struct that points at them.

    `model` is any object/dict with the fields of SURVEY 8(b) `nepzbl_params` (minus the list
    capacities and skin, which the oracle does not need).
    """

    def __init__(self, model: dict):
        m = dict(model)
        self.m = m
        f64 = lambda k: np.ascontiguousarray(np.asarray(m[k], dtype=np.float64))
        self.c_radial = f64("c_radial")
        self.c_angular = f64("c_angular")
        self.q_scaler = f64("q_scaler")
        self.w0 = f64("w0")
        self.b0 = f64("b0")
        self.w1 = f64("w1")
        self.atomic_number = f64("atomic_number")
        self.mass = f64("mass")
        s = _CParams()
        s.n_types = int(m["n_types"])
        s.rc_radial = float(m["rc_radial"]); s.rc_angular = float(m["rc_angular"])
        s.n_max_radial = int(m["n_max_radial"]); s.n_max_angular = int(m["n_max_angular"])
        s.basis_radial = int(m["basis_radial"]); s.basis_angular = int(m["basis_angular"])
        s.l_max = int(m["l_max"]); s.has_4body = int(m["has_4body"]); s.n_neurons = int(m["n_neurons"])
        s.has_5body = int(m.get("has_5body", 0))
        s.c_radial = _dp(self.c_radial); s.c_angular = _dp(self.c_angular)
        s.q_scaler = _dp(self.q_scaler)
        s.w0 = _dp(self.w0); s.b0 = _dp(self.b0); s.w1 = _dp(self.w1)
        s.b1 = float(m["b1"])
        s.zbl_enabled = int(m["zbl_enabled"])
        s.zbl_r_inner = float(m["zbl_r_inner"]); s.zbl_r_outer = float(m["zbl_r_outer"])
        nt = len(m["zbl_c"])
        assert nt <= 4 and len(m["zbl_d"]) == nt
        s.zbl_n_terms = nt
        for k in range(nt):
            s.zbl_c[k] = float(m["zbl_c"][k]); s.zbl_d[k] = float(m["zbl_d"][k])
        s.zbl_a_num = float(m["zbl_a_num"]); s.zbl_a_pow = float(m["zbl_a_pow"])
        s.coulomb_k = float(m["coulomb_k"])
        s.atomic_number = _dp(self.atomic_number); s.mass = _dp(self.mass)
        self.c = s
        self.D = lib().orc_descriptor_dim(C.byref(s))
        nt2 = s.n_types ** 2
        assert self.c_radial.size == nt2 * (s.n_max_radial + 1) * (s.basis_radial + 1)
        assert self.c_angular.size == nt2 * (s.n_max_angular + 1) * (s.basis_angular + 1)
        assert self.q_scaler.size == self.D and self.w0.size == s.n_neurons * self.D
        assert self.b0.size == s.n_neurons and self.w1.size == s.n_neurons

    @property
    def ref(self):
        return C.byref(self.c)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def zbl_pair(P: Params, r: float, ti: int = 0, tj: int = 0):
    """U_ZBL(r), dU/dr -- Eq. 2-4, switch."""
    u = C.c_double(); du = C.c_double()
    lib().orc_zbl_pair(P.ref, C.c_int(ti), C.c_int(tj), C.c_double(r), C.byref(u), C.byref(du))
    return u.value, du.value


def zbl_screening_length(P: Params, ti: int = 0, tj: int = 0) -> float:
    """a of Eq. 4."""
    return float(lib().orc_zbl_screening_length(P.ref, C.c_int(ti), C.c_int(tj)))


def radial_basis(r: float, rc: float, basis: int):
    """f_k(r), df_k/dr for k = 0..basis (S:B)."""
    f = np.zeros(basis + 1); df = np.zeros(basis + 1)
    lib().orc_radial_basis(C.c_double(r), C.c_double(rc), C.c_int(basis), _dp(f), _dp(df))
    return f, df


def radial_functions(P: Params, which: int, r: float, ti: int = 0, tj: int = 0):
    """g_n(r), dg_n/dr for the radial (which=0) or angular (which=1) channel (S:B)."""
    nmax = P.c.n_max_angular if which else P.c.n_max_radial
    g = np.zeros(nmax + 1); dg = np.zeros(nmax + 1)
    lib().orc_radial_functions(P.ref, C.c_int(which), C.c_int(ti), C.c_int(tj), C.c_double(r),
                               _dp(g), _dp(dg))
    return g, dg


def descriptor_site(P: Params, d: np.ndarray, ti: int = 0, tj=None, want_dq: bool = False):
    """q[D] (and dq[D][nn][3]) of one site given neighbour displacement vectors d[nn][3] (S:C)."""
    d = np.ascontiguousarray(d, dtype=np.float64).reshape(-1, 3)
    nn = d.shape[0]
    tj = np.zeros(nn, dtype=np.int32) if tj is None else np.ascontiguousarray(tj, dtype=np.int32)
    q = np.zeros(P.D)
    dq = np.zeros((P.D, max(nn, 1), 3)) if want_dq else None
    lib().orc_descriptor_site(P.ref, C.c_int(ti), C.c_int(nn), _ip(tj), _dp(d), _dp(q),
                              _dp(dq) if want_dq else None)
    return (q, dq[:, :nn]) if want_dq else q


def site_energy(P: Params, q: np.ndarray):
    """U^NEP(q), Fp = dU/dq (S:D)."""
    q = np.ascontiguousarray(q, dtype=np.float64)
    U = C.c_double(); Fp = np.zeros(P.D)
    lib().orc_site_energy(P.ref, _dp(q), C.byref(U), _dp(Fp))
    return U.value, Fp


def _sys_args(pos, types, box, pbc):
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    assert pos.ndim == 2 and pos.shape[0] == 3, "pos is SoA: shape (3, n)"
    n = pos.shape[1]
    types = np.zeros(n, dtype=np.int32) if types is None else np.ascontiguousarray(types, dtype=np.int32)
    box = np.ascontiguousarray(box, dtype=np.float64).reshape(9)
    pbc = np.ascontiguousarray(pbc, dtype=np.int32).reshape(3)
    return pos, n, types, box, pbc


def neighbors(pos, box, pbc, rc: float, use_cell: bool = False, cap: int = 256, want_d: bool = False, sel=None):
    """Neighbour lists (S:A): nn[n], nl[n][cap] (canonical order), optionally displacement vectors.
    sel: only these atoms (row t of the result belongs to atom sel[t])."""
    pos, n, _, box, pbc = _sys_args(pos, None, box, pbc)
    if sel is not None:
        assert not want_d
        sel = np.ascontiguousarray(sel, dtype=np.int32)
        nn = np.zeros(sel.size, dtype=np.int32)
        nl = np.full((sel.size, cap), -1, dtype=np.int32)
        f = lib().orc_neighbors_sel
        f.restype = C.c_int
        r = f(C.c_int(n), _dp(pos), _dp(box), _ip(pbc), C.c_double(rc), C.c_int(int(use_cell)), C.c_int(cap),
              C.c_int(sel.size), _ip(sel), _ip(nn), _ip(nl))
        if r < 0:
            raise RuntimeError(f"oracle neighbours failed: {r}")
        if r > cap:
            raise RuntimeError(f"oracle neighbour capacity {cap} < {r}")
        return nn, nl
    nn = np.zeros(n, dtype=np.int32)
    nl = np.full((n, cap), -1, dtype=np.int32)
    nd = np.zeros((n, cap, 3)) if want_d else None
    r = lib().orc_neighbors(C.c_int(n), _dp(pos), _dp(box), _ip(pbc), C.c_double(rc),
                            C.c_int(int(use_cell)), C.c_int(cap), _ip(nn), _ip(nl),
                            _dp(nd) if want_d else None)
    if r < 0:
        raise RuntimeError(f"oracle neighbours failed: {r}")
    if r > cap:
        raise RuntimeError(f"oracle neighbour capacity {cap} < {r}")
    return (nn, nl, nd) if want_d else (nn, nl)


@dataclass
class Result:
    energy: np.ndarray
    force: np.ndarray      # (3, n)
    virial: np.ndarray     # (9, n)
    q: np.ndarray | None = field(default=None)  # (n, D)


def compute(P: Params, pos, types, box, pbc, use_cell: bool | None = None, want_q: bool = False,
            sel=None, want_force: bool = True, want_virial: bool = True) -> Result:
    """Per-atom energy (Eq. 1), force and virial (S:E).  sel: evaluate only these atoms (others NaN)."""
    pos, n, types, box, pbc = _sys_args(pos, types, box, pbc)
    if use_cell is None:
        use_cell = n > 3000
    e = np.zeros(n)
    f = np.zeros((3, n)) if want_force else None
    w = np.zeros((9, n)) if want_virial else None
    q = np.zeros((n, P.D)) if want_q else None
    if sel is None:
        nsel, selp = -1, None
    else:
        sel = np.ascontiguousarray(sel, dtype=np.int32)
        nsel, selp = sel.size, _ip(sel)
    r = lib().orc_compute(P.ref, C.c_int(n), _dp(pos), _ip(types), _dp(box), _ip(pbc),
                          C.c_int(int(use_cell)), _dp(e), _dp(f) if want_force else None,
                          _dp(w) if want_virial else None, _dp(q) if want_q else None,
                          C.c_int(nsel), selp)
    if r != 0:
        raise RuntimeError(f"oracle compute failed: {r}")
    return Result(e, f, w, q)


def md_run(P: Params, pos, vel, types, box, pbc, nsteps: int, dt_max: float, max_disp: float,
           use_cell: bool | None = None):
    """nsteps of velocity-Verlet with the adaptive step of P:77 (S:F).  Returns new pos, vel and traces."""
    pos, n, types, box, pbc = _sys_args(pos, types, box, pbc)
    pos = pos.copy()
    vel = np.ascontiguousarray(vel, dtype=np.float64).copy()
    if use_cell is None:
        use_cell = n > 3000
    dt = np.zeros(max(nsteps, 1)); ep = np.zeros(nsteps + 1); ek = np.zeros(nsteps + 1)
    r = lib().orc_md_run(P.ref, C.c_int(n), _dp(pos), _dp(vel), _ip(types), _dp(box), _ip(pbc),
                         C.c_int(nsteps), C.c_double(dt_max), C.c_double(max_disp),
                         C.c_int(int(use_cell)), _dp(dt), _dp(ep), _dp(ek))
    if r != 0:
        raise RuntimeError(f"oracle md failed: {r}")
    return pos, vel, dt[:nsteps], ep, ek


KB_EV_PER_K = 8.617333262e-5


def nhc_half_step(M: int, nf: float, kT: float, tau: float, delta: float, ke2: float, xi, vxi):
    """One NHC(delta) operator (ref. [32]; DESIGN C-24) on copies of xi, vxi.  Returns s, xi, vxi."""
    xi = np.ascontiguousarray(xi, dtype=np.float64).copy()
    vxi = np.ascontiguousarray(vxi, dtype=np.float64).copy()
    f = lib().orc_nhc_half_step
    f.restype = C.c_double
    s = f(C.c_int(M), C.c_double(nf), C.c_double(kT), C.c_double(tau), C.c_double(delta), C.c_double(ke2),
          _dp(xi), _dp(vxi))
    return float(s), xi, vxi


def md_run_nhc(P: Params, pos, vel, types, box, pbc, nsteps: int, dt_max: float, max_disp: float,
               group, T: float, tau: float, chain: int = 4, xi=None, vxi=None, use_cell: bool | None = None):
    """md_run with a Nose-Hoover chain (ref. [32]) on the atoms with group != 0.
    Returns a dict: pos, vel, dt, epot, ekin, conserved, t_group, xi, vxi."""
    pos, n, types, box, pbc = _sys_args(pos, types, box, pbc)
    pos = pos.copy()
    vel = np.ascontiguousarray(vel, dtype=np.float64).copy()
    group = np.ascontiguousarray(group, dtype=np.uint8)
    assert group.size == n
    if use_cell is None:
        use_cell = n > 3000
    xi = np.zeros(chain) if xi is None else np.ascontiguousarray(xi, dtype=np.float64).copy()
    vxi = np.zeros(chain) if vxi is None else np.ascontiguousarray(vxi, dtype=np.float64).copy()
    dt = np.zeros(max(nsteps, 1)); ep = np.zeros(nsteps + 1); ek = np.zeros(nsteps + 1)
    cons = np.zeros(nsteps + 1); tg = np.zeros(nsteps + 1)
    f = lib().orc_md_run_nhc
    f.restype = C.c_int
    r = f(P.ref, C.c_int(n), _dp(pos), _dp(vel), _ip(types), _dp(box), _ip(pbc), C.c_int(nsteps),
          C.c_double(dt_max), C.c_double(max_disp), C.c_int(int(use_cell)),
          group.ctypes.data_as(C.POINTER(C.c_uint8)), C.c_double(T), C.c_double(tau), C.c_int(chain),
          _dp(xi), _dp(vxi), _dp(dt), _dp(ep), _dp(ek), _dp(cons), _dp(tg))
    if r != 0:
        raise RuntimeError(f"oracle md (nhc) failed: {r}")
    return dict(pos=pos, vel=vel, dt=dt[:nsteps], epot=ep, ekin=ek, conserved=cons, t_group=tg, xi=xi, vxi=vxi)


def wigner_seitz(site, pos, box, pbc, sel=None):
    """Wigner-Seitz occupancy (ref. [34]): nearest[n], occ[n_sites], (n_vacancies, n_interstitials).
    Brute force over all sites.  sel: only these atoms are assigned (others -1)."""
    site = np.ascontiguousarray(site, dtype=np.float64)
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    assert site.ndim == 2 and site.shape[0] == 3 and pos.ndim == 2 and pos.shape[0] == 3
    ns, n = site.shape[1], pos.shape[1]
    box = np.ascontiguousarray(box, dtype=np.float64).reshape(9)
    pbc = np.ascontiguousarray(pbc, dtype=np.int32).reshape(3)
    nearest = np.full(n, -1, dtype=np.int32)
    occ = np.zeros(ns, dtype=np.int32)
    counts = np.zeros(2, dtype=np.int64)
    if sel is None:
        nsel, selp = -1, None
    else:
        sel = np.ascontiguousarray(sel, dtype=np.int32)
        nsel, selp = sel.size, _ip(sel)
    f = lib().orc_wigner_seitz
    f.restype = C.c_int
    r = f(C.c_int(ns), _dp(site), C.c_int(n), _dp(pos), _dp(box), _ip(pbc), C.c_int(nsel), selp,
          _ip(nearest), _ip(occ), counts.ctypes.data_as(C.POINTER(C.c_int64)))
    if r != 0:
        raise RuntimeError(f"oracle wigner_seitz failed: {r}")
    return nearest, occ, (int(counts[0]), int(counts[1]))

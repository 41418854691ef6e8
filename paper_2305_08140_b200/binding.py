"""Thin Python binding of the C ABI in include/nepzbl.h (same names, argument marshalling only).

Every step of the path runs in the CUDA kernels of csrc/libnepzbl.so; this module only converts
torch tensors to device pointers.  PyTorch is used for device memory and streams, nothing else.
If the library is missing the import FAILS LOUDLY -- there is no CPU or PyTorch fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# NEPZBL_LIB=checked: the bounds-checked build of the same sources (build.py, common.cuh NZ_CHECK)
LIB_PATH = os.path.join(_HERE, "csrc", "libnepzbl_checked.so" if os.environ.get("NEPZBL_LIB") == "checked" else "libnepzbl.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2305_08140_b200.build` "
                      "(nvcc, sm_100a). There is no fallback path.")
_lib = C.CDLL(LIB_PATH)

OK = 0
ERRORS = {-1: "INVALID_ARG", -2: "BOX_NOT_ORTHOGONAL", -3: "BOX_TOO_SMALL", -4: "NEIGHBOR_OVERFLOW",
          -5: "NONFINITE", -6: "CUDA", -7: "UNSUPPORTED", -8: "WORKSPACE", -9: "STATE"}

EXPORTS = ["nep_zbl_create", "nep_zbl_destroy", "nep_zbl_last_error", "nep_zbl_descriptor_dim",
           "nep_zbl_workspace_bytes", "nep_zbl_set_workspace", "neighbor_build", "neighbor_get",
           "nep_zbl_compute", "nep_zbl_compute_host", "nep_zbl_get_descriptors", "md_init", "md_step",
           "md_run", "md_step_host", "md_request_rebuild", "md_energies", "md_get_forces", "md_get_counters",
           "md_set_thermostat", "md_get_thermostat", "md_set_thermostat_state", "wigner_seitz_set_reference", "wigner_seitz_count",
           "nep_zbl_uses_graph", "nep_zbl_network_mode", "nep_zbl_last_counts", "nep_zbl_launch_count", "nep_zbl_profile", "nep_zbl_profile_read", "nep_zbl_ffma_peak",
           "nep_zbl_energy_sums_static"]
PROFILE_SLOTS = ["integrate_a", "rebuild", "k_radial", "k_angular_nn", "k_force", "k_zbl", "kick_b", "k_site_fp64"]


class NepZblError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"NEPZBL_E_{ERRORS.get(code, code)}: {msg}")
        self.code = code


class _CParams(C.Structure):
    _fields_ = [
        ("n_types", C.c_int32),
        ("rc_radial", C.c_double), ("rc_angular", C.c_double),
        ("n_max_radial", C.c_int32), ("n_max_angular", C.c_int32),
        ("basis_radial", C.c_int32), ("basis_angular", C.c_int32),
        ("l_max", C.c_int32), ("has_4body", C.c_int32), ("has_5body", C.c_int32), ("n_neurons", C.c_int32),
        ("c_radial", C.c_void_p), ("c_angular", C.c_void_p), ("q_scaler", C.c_void_p),
        ("w0", C.c_void_p), ("b0", C.c_void_p), ("w1", C.c_void_p),
        ("b1", C.c_double),
        ("zbl_enabled", C.c_int32),
        ("zbl_r_inner", C.c_double), ("zbl_r_outer", C.c_double),
        ("zbl_n_terms", C.c_int32),
        ("zbl_c", C.c_double * 4), ("zbl_d", C.c_double * 4),
        ("zbl_a_num", C.c_double), ("zbl_a_pow", C.c_double), ("coulomb_k", C.c_double),
        ("atomic_number", C.c_void_p), ("mass", C.c_void_p),
        ("skin", C.c_double),
        ("cap_radial", C.c_int32), ("cap_angular", C.c_int32),
    ]


_vp, _i64, _i32, _dbl, _sz = C.c_void_p, C.c_int64, C.c_int32, C.c_double, C.c_size_t
_lib.nep_zbl_create.argtypes = [C.POINTER(_CParams), C.c_int, _vp, C.POINTER(_vp)]
_lib.nep_zbl_create.restype = C.c_int
_lib.nep_zbl_destroy.argtypes = [_vp]
_lib.nep_zbl_destroy.restype = None
_lib.nep_zbl_last_error.argtypes = [_vp]
_lib.nep_zbl_last_error.restype = C.c_char_p
_lib.nep_zbl_descriptor_dim.argtypes = [_vp]
_lib.nep_zbl_descriptor_dim.restype = C.c_int
_lib.nep_zbl_workspace_bytes.argtypes = [_vp, _i64]
_lib.nep_zbl_workspace_bytes.restype = _sz
_lib.nep_zbl_set_workspace.argtypes = [_vp, _vp, _sz, _i64]
_lib.nep_zbl_set_workspace.restype = C.c_int
_lib.neighbor_build.argtypes = [_vp, _i64, _vp, _vp, C.POINTER(_dbl), C.POINTER(_i32)]
_lib.neighbor_build.restype = C.c_int
_lib.neighbor_get.argtypes = [_vp, C.c_int, _vp, _vp]
_lib.neighbor_get.restype = C.c_int
for _f in (_lib.nep_zbl_compute, _lib.nep_zbl_compute_host):
    _f.argtypes = [_vp, _i64, _vp, _vp, C.POINTER(_dbl), C.POINTER(_i32), _vp, _vp, _vp]
    _f.restype = C.c_int
_lib.nep_zbl_get_descriptors.argtypes = [_vp, _vp]
_lib.nep_zbl_get_descriptors.restype = C.c_int
_lib.md_init.argtypes = [_vp, _i64, _vp, _vp, _vp, C.POINTER(_dbl), C.POINTER(_i32)]
_lib.md_init.restype = C.c_int
_lib.md_step.argtypes = [_vp, _dbl, _dbl, C.POINTER(_dbl), C.POINTER(_i32)]
_lib.md_step.restype = C.c_int
_lib.md_run.argtypes = [_vp, _i64, _dbl, _dbl, _vp, C.POINTER(_i64)]
_lib.md_run.restype = C.c_int
_lib.md_step_host.argtypes = [_vp, _vp, _vp, _dbl, _dbl, C.POINTER(_dbl), C.POINTER(_i32)]
_lib.md_step_host.restype = C.c_int
_lib.md_request_rebuild.argtypes = [_vp]
_lib.md_request_rebuild.restype = C.c_int
_lib.md_energies.argtypes = [_vp, C.POINTER(_dbl), C.POINTER(_dbl)]
_lib.md_energies.restype = C.c_int
_lib.md_get_forces.argtypes = [_vp, _vp, _vp]
_lib.md_get_forces.restype = C.c_int
_lib.md_get_counters.argtypes = [_vp, C.POINTER(_i64), C.POINTER(_i64), C.POINTER(_i64)]
_lib.md_get_counters.restype = C.c_int
_lib.md_set_thermostat.argtypes = [_vp, _vp, C.c_double, C.c_double, C.c_int32]
_lib.md_set_thermostat.restype = C.c_int
_lib.md_get_thermostat.argtypes = [_vp, C.POINTER(_dbl), C.POINTER(_dbl), C.POINTER(_dbl), C.POINTER(_dbl)]
_lib.md_get_thermostat.restype = C.c_int
_lib.md_set_thermostat_state.argtypes = [_vp, C.POINTER(_dbl), C.POINTER(_dbl)]
_lib.md_set_thermostat_state.restype = C.c_int
_lib.wigner_seitz_set_reference.argtypes = [_vp, _i64, _vp, C.POINTER(_dbl), C.POINTER(_i32)]
_lib.wigner_seitz_set_reference.restype = C.c_int
_lib.wigner_seitz_count.argtypes = [_vp, _i64, _vp, _vp, _vp, C.POINTER(_i64), C.POINTER(_i64)]
_lib.wigner_seitz_count.restype = C.c_int
_lib.nep_zbl_uses_graph.argtypes = [_vp]
_lib.nep_zbl_uses_graph.restype = C.c_int
_lib.nep_zbl_network_mode.argtypes = [_vp]
_lib.nep_zbl_network_mode.restype = C.c_int
_lib.nep_zbl_last_counts.argtypes = [_vp, C.POINTER(_i64), C.POINTER(_i64)]
_lib.nep_zbl_last_counts.restype = C.c_int
_lib.nep_zbl_launch_count.argtypes = [_vp]
_lib.nep_zbl_launch_count.restype = _i64
_lib.nep_zbl_profile.argtypes = [_vp, C.c_int]
_lib.nep_zbl_profile.restype = C.c_int
_lib.nep_zbl_profile_read.argtypes = [_vp, C.POINTER(_dbl), C.POINTER(_i64)]
_lib.nep_zbl_profile_read.restype = C.c_int
_lib.nep_zbl_ffma_peak.argtypes = [_vp, C.POINTER(_dbl)]
_lib.nep_zbl_ffma_peak.restype = C.c_int
_lib.nep_zbl_energy_sums_static.argtypes = [_i64, _vp, _vp, _vp, _i32, C.POINTER(_dbl), _vp, _vp, C.c_char_p, _sz]
_lib.nep_zbl_energy_sums_static.restype = C.c_int
STATIC_MAX_ATOMS = 33554432   # NEPZBL_STATIC_MAX_ATOMS


def _ptr(t):
    if t is None:
        return None
    if isinstance(t, torch.Tensor):
        assert t.is_contiguous()
        return t.data_ptr()
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return t.ctypes.data
    raise TypeError(type(t))


def nep_zbl_energy_sums_static(vel, energy, types, mass, out, stream=None, n_atoms=None):
    """{E_pot, E_kin} into `out` (2 doubles on the device) without any allocation: include/nepzbl.h.  Asynchronous;
    `mass` is a host sequence of one value per type; `n_atoms` defaults to len(energy)."""
    n = int(energy.numel() if n_atoms is None else n_atoms)
    m = (C.c_double * len(mass))(*[float(x) for x in mass])
    err = C.create_string_buffer(256)
    rc = _lib.nep_zbl_energy_sums_static(n, _ptr(vel), _ptr(energy), _ptr(types), len(mass), m, _ptr(out),
                                         stream.cuda_stream if stream is not None else None, err, len(err))
    if rc != OK:
        raise NepZblError(rc, err.value.decode())
    return out


def _box(box):
    return (C.c_double * 9)(*[float(x) for x in np.asarray(box, dtype=np.float64).reshape(9)])


def _pbc(pbc):
    return (C.c_int32 * 3)(*[int(x) for x in np.asarray(pbc).reshape(3)])


class NepZbl:
    """Owns one nepzbl_handle plus its torch-allocated workspace.  Method names = C entry points."""

    def __init__(self, model: dict, n_atoms: int, device: int = 0, stream: torch.cuda.Stream | None = None):
        m = model
        self._keep = {}
        f64 = lambda k: self._keep.setdefault(k, np.ascontiguousarray(np.asarray(m[k], dtype=np.float64)))
        p = _CParams()
        p.n_types = int(m["n_types"])
        p.rc_radial = float(m["rc_radial"]); p.rc_angular = float(m["rc_angular"])
        p.n_max_radial = int(m["n_max_radial"]); p.n_max_angular = int(m["n_max_angular"])
        p.basis_radial = int(m["basis_radial"]); p.basis_angular = int(m["basis_angular"])
        p.l_max = int(m["l_max"]); p.has_4body = int(m["has_4body"]); p.n_neurons = int(m["n_neurons"])
        p.has_5body = int(m.get("has_5body", 0))
        for k in ("c_radial", "c_angular", "q_scaler", "w0", "b0", "w1", "atomic_number", "mass"):
            setattr(p, k, f64(k).ctypes.data)
        p.b1 = float(m["b1"])
        p.zbl_enabled = int(m["zbl_enabled"])
        p.zbl_r_inner = float(m["zbl_r_inner"]); p.zbl_r_outer = float(m["zbl_r_outer"])
        p.zbl_n_terms = len(m["zbl_c"])
        for k in range(p.zbl_n_terms):
            p.zbl_c[k] = float(m["zbl_c"][k]); p.zbl_d[k] = float(m["zbl_d"][k])
        p.zbl_a_num = float(m["zbl_a_num"]); p.zbl_a_pow = float(m["zbl_a_pow"])
        p.coulomb_k = float(m["coulomb_k"])
        p.skin = float(m["skin"]); p.cap_radial = int(m["cap_radial"]); p.cap_angular = int(m["cap_angular"])
        self.cap_radial, self.cap_angular = p.cap_radial, p.cap_angular
        self.device = torch.device("cuda", device)
        self.stream = stream
        h = _vp()
        rc = _lib.nep_zbl_create(C.byref(p), device, _vp(stream.cuda_stream if stream else 0), C.byref(h))
        if rc != OK:
            raise NepZblError(rc, _lib.nep_zbl_last_error(None).decode())
        self.h = h
        self.D = _lib.nep_zbl_descriptor_dim(self.h)
        self.n_cap = int(n_atoms)
        nbytes = _lib.nep_zbl_workspace_bytes(self.h, self.n_cap)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        off = (-self.workspace.data_ptr()) % 256
        self._chk(_lib.nep_zbl_set_workspace(self.h, self.workspace.data_ptr() + off, nbytes, self.n_cap))
        self.workspace_bytes = nbytes

    def _chk(self, rc):
        if rc != OK:
            raise NepZblError(rc, _lib.nep_zbl_last_error(self.h).decode())

    def close(self):
        if getattr(self, "h", None):
            _lib.nep_zbl_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- C entry points
    def neighbor_build(self, pos, types, box, pbc):
        self._n = pos.shape[-1]
        self._chk(_lib.neighbor_build(self.h, self._n, _ptr(pos), _ptr(types), _box(box), _pbc(pbc)))

    def neighbor_get(self, which: int):
        cap = self.cap_angular if which else self.cap_radial
        nn = torch.empty(self._n, dtype=torch.int32, device=self.device)
        nl = torch.empty((self._n, cap), dtype=torch.int32, device=self.device)
        self._chk(_lib.neighbor_get(self.h, which, _ptr(nn), _ptr(nl)))
        return nn, nl

    def nep_zbl_compute(self, pos, types, box, pbc, energy=None, force=None, virial=None):
        self._n = pos.shape[-1]
        self._chk(_lib.nep_zbl_compute(self.h, self._n, _ptr(pos), _ptr(types), _box(box), _pbc(pbc),
                                       _ptr(energy), _ptr(force), _ptr(virial)))

    def nep_zbl_compute_host(self, pos, types, box, pbc, energy=None, force=None, virial=None):
        self._n = pos.shape[-1]
        self._chk(_lib.nep_zbl_compute_host(self.h, self._n, _ptr(pos), _ptr(types), _box(box), _pbc(pbc),
                                            _ptr(energy), _ptr(force), _ptr(virial)))

    def nep_zbl_get_descriptors(self):
        q = torch.empty((self._n, self.D), dtype=torch.float32, device=self.device)
        self._chk(_lib.nep_zbl_get_descriptors(self.h, _ptr(q)))
        return q

    def md_init(self, pos, vel, types, box, pbc):
        self._n = pos.shape[-1]
        self._md_keep = (pos, vel, types)      # the library integrates these buffers in place
        self._chk(_lib.md_init(self.h, self._n, _ptr(pos), _ptr(vel), _ptr(types), _box(box), _pbc(pbc)))

    def md_step(self, dt_max: float, max_displacement: float):
        dt = _dbl(); rb = _i32()
        self._chk(_lib.md_step(self.h, dt_max, max_displacement, C.byref(dt), C.byref(rb)))
        return dt.value, rb.value

    def md_run(self, n_steps: int, dt_max: float, max_displacement: float, want_trace: bool = False):
        tr = np.zeros(max(n_steps, 1)) if want_trace else None
        nr = _i64()
        self._chk(_lib.md_run(self.h, n_steps, dt_max, max_displacement, _ptr(tr), C.byref(nr)))
        return (tr[:n_steps] if want_trace else None), nr.value

    def md_step_host(self, pos_host, vel_host, dt_max: float, max_displacement: float):
        dt = _dbl(); rb = _i32()
        self._chk(_lib.md_step_host(self.h, _ptr(pos_host), _ptr(vel_host), dt_max, max_displacement,
                                    C.byref(dt), C.byref(rb)))
        return dt.value, rb.value

    def md_request_rebuild(self):
        self._chk(_lib.md_request_rebuild(self.h))

    def md_energies(self):
        ep = _dbl(); ek = _dbl()
        self._chk(_lib.md_energies(self.h, C.byref(ep), C.byref(ek)))
        return ep.value, ek.value

    def md_get_forces(self):
        f = torch.empty((3, self._n), dtype=torch.float32, device=self.device)
        e = torch.empty(self._n, dtype=torch.float64, device=self.device)
        self._chk(_lib.md_get_forces(self.h, _ptr(f), _ptr(e)))
        return f, e

    def md_get_counters(self):
        a = _i64(); b = _i64(); c = _i64()
        self._chk(_lib.md_get_counters(self.h, C.byref(a), C.byref(b), C.byref(c)))
        return a.value, b.value, c.value

    def md_set_thermostat(self, group, temperature: float, tau: float, chain_length: int = 4):
        """group: uint8 device tensor [n] (non-zero = thermostatted) or None to switch off."""
        self._group_keep = group
        self._chain = chain_length
        self._chk(_lib.md_set_thermostat(self.h, _ptr(group), temperature, tau, chain_length))

    def md_set_thermostat_state(self, xi, vxi):
        m = self._chain
        a = (_dbl * 8)(*[float(x) for x in xi[:m]]); b = (_dbl * 8)(*[float(x) for x in vxi[:m]])
        self._chk(_lib.md_set_thermostat_state(self.h, a, b))

    def md_get_thermostat(self):
        xi = (_dbl * 8)(); vxi = (_dbl * 8)(); tg = _dbl(); ex = _dbl()
        self._chk(_lib.md_get_thermostat(self.h, xi, vxi, C.byref(tg), C.byref(ex)))
        m = self._chain
        return np.array(xi[:m]), np.array(vxi[:m]), tg.value, ex.value

    def wigner_seitz_set_reference(self, site, box, pbc):
        """site: fp64 device tensor (3, n_sites)."""
        self._ws_ns = site.shape[-1]
        self._chk(_lib.wigner_seitz_set_reference(self.h, self._ws_ns, _ptr(site), _box(box), _pbc(pbc)))

    def wigner_seitz_count(self, pos, want_nearest: bool = True, want_occupancy: bool = True):
        """pos: fp64 device tensor (3, n).  Returns nearest (n,), occupancy (n_sites,), (n_vac, n_sia)."""
        n = pos.shape[-1]
        nearest = torch.empty(n, dtype=torch.int32, device=self.device) if want_nearest else None
        occ = torch.empty(self._ws_ns, dtype=torch.int32, device=self.device) if want_occupancy else None
        nv = _i64(); ni = _i64()
        self._chk(_lib.wigner_seitz_count(self.h, n, _ptr(pos), _ptr(nearest), _ptr(occ), C.byref(nv), C.byref(ni)))
        return nearest, occ, (nv.value, ni.value)

    def nep_zbl_uses_graph(self) -> bool:
        return bool(_lib.nep_zbl_uses_graph(self.h))

    def nep_zbl_network_mode(self) -> int:
        return int(_lib.nep_zbl_network_mode(self.h))

    def nep_zbl_last_counts(self):
        a = _i64(); b = _i64()
        self._chk(_lib.nep_zbl_last_counts(self.h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def nep_zbl_launch_count(self) -> int:
        return int(_lib.nep_zbl_launch_count(self.h))

    def nep_zbl_profile(self, enable: bool):
        self._chk(_lib.nep_zbl_profile(self.h, int(enable)))

    def nep_zbl_profile_read(self):
        ms = (_dbl * 8)(); cnt = (_i64 * 8)()
        self._chk(_lib.nep_zbl_profile_read(self.h, ms, cnt))
        return {k: (ms[i], cnt[i]) for i, k in enumerate(PROFILE_SLOTS)}

    def nep_zbl_ffma_peak(self) -> float:
        t = _dbl()
        self._chk(_lib.nep_zbl_ffma_peak(self.h, C.byref(t)))
        return t.value

    # ---- convenience (marshalling only)
    def compute(self, pos_np, types_np, box, pbc, virial: bool = True):
        """numpy in / numpy out through device tensors (nep_zbl_compute)."""
        n = pos_np.shape[1]
        pos = torch.from_numpy(np.ascontiguousarray(pos_np)).to(self.device)
        types = torch.from_numpy(np.ascontiguousarray(types_np, dtype=np.int32)).to(self.device)
        e = torch.empty(n, dtype=torch.float64, device=self.device)
        f = torch.empty((3, n), dtype=torch.float32, device=self.device)
        w = torch.empty((9, n), dtype=torch.float32, device=self.device) if virial else None
        self.nep_zbl_compute(pos, types, box, pbc, e, f, w)
        return e.cpu().numpy(), f.cpu().numpy(), (w.cpu().numpy() if virial else None)

"""bench.py -- atom-steps/s of the NEP-ZBL MD hot path on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference] [--workload config2]

One "step" = one velocity-Verlet step of the whole hot path (S1-S8 of DESIGN.md: integrator half
kicks + drift, list rebuild when the skin is exhausted, radial/angular descriptors, network,
force back-pass, ZBL).  BASELINE.json's metric names no config, so the default workload is the largest
single-GPU configuration, configs[3] ("config4"): the 8 192 000-atom bulk cascade (160^3 bcc cells, 300 K,
100 keV PKA, adaptive time step); the other configs are timed in the same run and reported under `per_config`.
The cascade configs rebuild their list once per ~60 steps; so that S2 is inside a timed region of any length, ONE
rebuild is requested at the start of every cascade config's timed steps (config.forced_rebuilds) -- at --steps 20
that over-represents the rebuild (conservative).
Prints ONE JSON line (rank 0).  Keys: see DESIGN.md "Measurement".

  value      K steps enqueued back to back by md_run (no host round trip), state resident in HBM,
             timed with CUDA events on the launch stream, barrier + synchronize on both sides,
             max over ranks.  `config.l2` says how the L2 rule is met.
  e2e        the same steps through md_step_host: pos/vel copied host->device and device->host
             every step from/to pinned host buffers, inside the timed region.
  roofline   dominant kernel: algorithmic flops (DESIGN.md table) / CUDA-event duration per launch.
  cpu_baseline  the fp64 oracle (oracle/, as it stands) timed on this box's host cores on a bounded
             sample of the same workload (rank 0, N = 1 only).
  --impl reference   times the oracle instead (this tier's reference arm); no GPU is touched.

Multi-GPU: the path does not shard (north_star: one GPU, no collectives) -> "replicas only":
every rank runs an independent replica (seed + rank) on its own GPU; value = sum of atom-steps
over ranks / max time over ranks; scaling = "weak".
"""
from __future__ import annotations

import argparse
import datetime
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "atom_steps_per_s"
UNIT = "atom-steps/s"
L2_BYTES = 126 * 1024 * 1024

# Algorithmic FP32 work per atom-step of each force kernel for the configs' model (5+5 radial
# functions, 9 basis functions, 24 (l,m), D = 30, 50 neurons) on bcc W at a = 3.165 A
# (58 radial / 14 angular neighbours inside the cutoffs, 88 / 26 list entries with the 1 A skin).
# Derivation: DESIGN.md "Algorithmic work per atom-step".  FMA = 2 flop.
# Per step of the path (S3, S4, S6, S7a = angular back-pass, S7r = radial back-pass + angular gather):
STEP_FLOP = {"S3": 3.2e3, "S4": 6.7e3, "S6": 6.6e3, "S7a": 14.0e3, "S7r": 8.6e3}
KERNEL_STEPS = {"k_radial": ("S3",), "k_angular_nn": ("S4", "S6", "S7a"), "k_force": ("S7r",)}
FLOP_PER_ATOM = {k: sum(STEP_FLOP[s] for s in v) for k, v in KERNEL_STEPS.items()}
# The same count for the paper-sized model (workload "paper": n_max 15/10, 100 neurons, no 4-body; DESIGN.md
# section 10): S3 58 x 51 + 240 + 16*9*2; S4 14 x (91 + 11*9*2 + 11*24*2) + 0.8k; S6 100 x (60*4 + 11);
# S7a 14 x (324 + 11*17*2 + 2*11*24*2) + 0.5k; S7r 58 x 142 + 16*9*2 + 0.2k
PAPER_STEP_FLOP = {"S3": 3.5e3, "S4": 12.2e3, "S6": 25.1e3, "S7a": 25.1e3, "S7r": 8.7e3}
PAPER_FLOP_PER_ATOM = {k: sum(PAPER_STEP_FLOP[s] for s in v) for k, v in KERNEL_STEPS.items()}
MODEL_DESC = {
    "alloy": "NEP-ZBL n_max 4/4, basis 8/8, l_max 4 + 4-body, 50 neurons, TWO atom types (W / Mo, type-pair tables), universal ZBL",
    "paper": "NEP-ZBL at the paper's sizes: n_max 15/10, basis 8/8, l_max 4, 100 neurons, rc 6/4 A, ZBL Eq. 3 refit 1-2 A "
             "(seeded random weights; a = 3.185 A)",
}
DEFAULT_MODEL_DESC = "NEP-ZBL n_max 4/4, basis 8/8, l_max 4 + 4-body, 50 neurons, rc 6/4 A, universal ZBL 1-2 A"
# Compulsory HBM bytes per atom-step of each kernel group (same table)
# (k_force carries the second half-kick: + 48 B of fp64 velocities; the per-atom record is 32 B)
BYTES_PER_ATOM = {"integrate_a": 152.0, "k_radial": 292.0, "k_angular_nn": 596.0, "k_force": 1168.0}
FP32_LANES_PER_SM = 128
# Wigner-Seitz count, compulsory HBM bytes per atom (one site per atom): position 24 + nearest 4 + occupancy
# read-modify-write 8 + count read 4 + cell-sorted site record 28 (the 27-cell scan re-reads sites from L1/L2)
WS_BYTES_PER_ATOM = 68.0
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` capture named in
# "source", valid for the kernel sources whose hash is "csrc_sha16" (csrc_sha16() below): when the kernels have
# changed since the capture, roofline.traffic is null and roofline.traffic_note says so.
NCU_TRAFFIC = {"csrc_sha16": "3da639d5ac0e32e3", "source": "profiles/r2_ncu_full.md", "bytes": {
    "config4": {"k_radial": 4389.4e6, "k_angular_nn": 6517.9e6, "k_force": 7150.9e6, "integrate_a": 1193.4e6},
    "config2": {"k_radial": 36.3e6, "k_angular_nn": 58.9e6, "k_force": 102.3e6, "integrate_a": 10.8e6},
    "paper": {"k_radial": 37.0e6, "k_angular_nn": 75.4e6, "k_force": 107.6e6}}}


def csrc_sha16() -> str:
    """Hash of everything the kernels are built from (csrc/*.cu, *.cuh and the C header)."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2305_08140_b200", "csrc")
    files = sorted(os.path.join(d, f) for f in os.listdir(d) if f.endswith((".cu", ".cuh")))
    for f in files + [os.path.join(ROOT, "include", "nepzbl.h")]:
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic(workload: str, kernel: str, cells):
    if cells is not None:
        return None, "non-standard cell count"
    if NCU_TRAFFIC["csrc_sha16"] != csrc_sha16():
        return None, f"stale: kernels changed since the capture in {NCU_TRAFFIC['source']}"
    v = NCU_TRAFFIC["bytes"].get(workload, {}).get(kernel)
    return v, (NCU_TRAFFIC["source"] if v is not None else "no capture for this workload")


def _dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def make_workload(name: str, seed_offset: int = 0, cells=None):
    from paper_2305_08140_b200 import workloads as wl
    if name == "config2":
        return wl.config2(seed=2 + seed_offset, cells=cells or 40)
    if name == "config3":
        return wl.config3(seed=3 + seed_offset, cells=cells or 80)
    if name == "config4":
        return wl.config4(seed=4 + seed_offset, cells=cells or 160)
    if name == "config5":
        return wl.config5(seed=5 + seed_offset, cells=cells or (160, 160, 100))
    if name == "alloy":   # config2's system with two atom types (W / Mo labels drawn 50/50)
        w = wl.config2(seed=2 + seed_offset, cells=cells or 40, model=wl.alloy_model(spread=0.05, stream=13))
        w.types = wl.random_types(w.n, 2 + seed_offset)
        return w
    if name == "paper":   # paper-sized model, a = 3.185 A, 0.01 A per step
        return wl.paper_bulk(cells or 40, seed=12 + seed_offset)
    raise SystemExit(f"unknown workload {name}")


# ------------------------------------------------------------------------------ clocks

class ClockSampler:
    """nvidia-smi sampled every 100 ms in the background; summarise the samples inside a window."""
    FIELDS = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(gpu_index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            p = [x.strip() for x in line.split(",")]
            if len(p) < 8:
                continue
            try:
                ts = datetime.datetime.strptime(p[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                self.rows.append((ts, float(p[1]), float(p[2]), float(p[3]), p[4], p[5], p[6], p[7]))
            except ValueError:
                continue

    def wait_first(self, timeout=5.0):
        t0 = time.time()
        while self.proc and not self.rows and time.time() - t0 < timeout:
            time.sleep(0.05)

    def stop(self):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except subprocess.TimeoutExpired:
                self.proc.kill()

    def summary(self, t0: float, t1: float) -> dict:
        rows = [r for r in self.rows if t0 - 0.05 <= r[0] <= t1 + 0.05] or self.rows[-3:]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        reasons = []
        for k, name in ((4, "hw_slowdown"), (5, "hw_thermal_slowdown"), (6, "sw_thermal_slowdown"), (7, "sw_power_cap")):
            if any(r[k] == "Active" for r in rows):
                reasons.append(name)
        return {"sm_mhz": float(np.median([r[1] for r in rows])), "sm_max_mhz": rows[0][2],
                "power_w_max": max(r[3] for r in rows), "samples": len(rows), "reasons": reasons}


# ------------------------------------------------------------------------------ oracle legs

CASCADE = {"config3": 1.0e4, "config4": 1.0e5, "config5": 1.0e5}     # PKA energies (eV) of the cascade configs


def sample_workload(name: str, cells: int):
    """The workload's own recipe at a smaller cell count (for the oracle legs: its cost is linear in N)."""
    from paper_2305_08140_b200 import workloads as wl
    if name in ("config3", "config4"):
        return wl.bulk_cascade(cells, CASCADE[name], seed=3 if name == "config3" else 4, n_steps=0, name=name)
    if name == "config5":
        return wl.config5(seed=5, cells=(cells, cells, max(4, cells * 5 // 8)))
    if name == "paper":
        return wl.paper_bulk(cells, seed=12)
    if name == "alloy":
        w = wl.config2(seed=2, cells=cells, model=wl.alloy_model(spread=0.05, stream=13))
        w.types = wl.random_types(w.n, 2)
        return w
    return wl.config2(seed=2, cells=cells)


def oracle_md_rate(workload_name: str, n_steps: int | None, warmup: int, budget_s: float):
    """Time the fp64 oracle's own MD loop (oracle.md_run, as it stands) on a bounded sample of the workload: the
    same recipe (lattice, temperature, PKA, model, dt rule) at the largest cell count from (6 ... 40)^3 whose run
    fits `budget_s`.  n_steps = None (the cpu_baseline leg): as many steps as fit the budget at 40^3 cells (fewer
    cells if not even 3 steps fit).  Cost is linear in N, so atom-steps/s carries over."""
    import oracle
    from paper_2305_08140_b200 import workloads as wl
    w = wl.thermal_bulk(10, seed=2, model=sample_workload(workload_name, 6).model)
    P = oracle.Params(w.model)
    oracle.md_run(P, w.pos, w.vel, w.types, w.box, w.pbc, 1, 1.0, np.inf)      # loads the library, spins up OpenMP
    t = time.perf_counter()
    oracle.md_run(P, w.pos, w.vel, w.types, w.box, w.pbc, 2, 1.0, np.inf)
    rate = 3 * w.n / (time.perf_counter() - t)                                 # atom-evaluations/s (3 evaluations)
    fits = lambda c, k: (warmup + k + 2) * 2 * c ** 3 / rate <= budget_s
    cells = 6
    for c in (8, 10, 12, 16, 24, 40):
        if fits(c, 3 if n_steps is None else n_steps):
            cells = c
    if n_steps is None:
        n_steps = int(max(3, min(200, budget_s * rate / (2 * cells ** 3) - 1)))
    w = sample_workload(workload_name, cells)
    pos, vel = w.pos, w.vel
    if warmup > 0:
        pos, vel, *_ = oracle.md_run(P, pos, vel, w.types, w.box, w.pbc, warmup, w.dt_max, w.max_displacement)
    t = time.perf_counter()
    oracle.md_run(P, pos, vel, w.types, w.box, w.pbc, n_steps, w.dt_max, w.max_displacement)
    dt = time.perf_counter() - t
    # md_run evaluates forces once before the loop: n_steps + 1 evaluations for n_steps steps
    return {"value": n_steps * w.n / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"{w.n} atoms of the {workload_name} recipe ({cells}^3-cell box instead of the full one), "
                      f"{n_steps} oracle MD steps (fp64, OpenMP, {n_steps + 1} force evaluations) in {dt:.1f} s"}, dt


def oracle_single_evaluations():
    """SURVEY 8(d) CPU-baseline item (i): ONE timed oracle evaluation (energy, force, virial) of config 1 and of
    config 2's initial state."""
    import oracle
    from paper_2305_08140_b200 import workloads as wl
    out = {}
    for name, w in (("config1", wl.config1()), ("config2_initial_state", wl.config2())):
        P = oracle.Params(w.model)
        t = time.perf_counter()
        oracle.compute(P, w.pos, w.types, w.box, w.pbc)
        dt = time.perf_counter() - t
        out[name] = {"atoms": w.n, "seconds": dt, "atoms_per_s": w.n / dt}
    return out


def run_reference(args):
    rank, _, world = _dist_env()
    if rank != 0:
        return 0
    cb, dt = oracle_md_rate(args.workload, args.steps, args.warmup, budget_s=150.0)
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": args.workload},
            "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------ B200 arm

def aggregate_max(ms_local: float, world: int, device=None) -> float:
    """max over ranks of a local duration (torch.distributed all-reduce; identity when world == 1)."""
    if world == 1:
        return ms_local
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_sum(x: float, world: int, device=None) -> float:
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def run_b200(args):
    import torch
    rank, local_rank, world = _dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the B200 arm has no CPU fallback (use --impl reference for the oracle)")
    from paper_2305_08140_b200 import build as cuda_build
    cuda_build.build()
    from paper_2305_08140_b200 import binding
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    stream = torch.cuda.Stream(device=dev)
    K, W = args.steps, args.warmup

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize(dev)

    sampler = ClockSampler(local_rank) if rank == 0 else None
    if sampler:
        sampler.wait_first()

    class Run:
        """One workload resident on the device: handle, state, and the timed legs."""

        def __init__(self, name, cells=None):
            self.name = name
            self.w = w = make_workload(name, seed_offset=rank, cells=cells)
            self.n = w.n
            self.cascade = name in CASCADE
            self.g = binding.NepZbl(w.model, w.n, device=local_rank, stream=stream)
            self.types = torch.from_numpy(w.types).to(dev)
            self.pos = self.vel = None

        def fresh_state(self):
            w = self.w
            self.pos = torch.from_numpy(w.pos.copy()).to(dev)
            self.vel = torch.from_numpy(w.vel.copy()).to(dev)
            self.g.md_init(self.pos, self.vel, self.types, w.box, w.pbc)

        def timed_steps(self):
            """W warm-up steps, then K steps back to back (md_run: no host round trip), CUDA events on the launch
            stream, barrier + synchronize on both sides; max over ranks."""
            g, w = self.g, self.w
            self.fresh_state()
            e0 = sum(g.md_energies())
            g.md_run(W, w.dt_max, w.max_displacement)
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            barrier()
            l0 = g.nep_zbl_launch_count()
            reb0 = g.md_get_counters()[1]
            forced = 0
            if self.cascade:            # S2 inside the timed region whatever K is (see the module docstring)
                g.md_request_rebuild()
                forced = 1
            t0 = time.time()
            ev0.record(stream)
            g.md_run(K, w.dt_max, w.max_displacement)
            ev1.record(stream)
            barrier()
            t1 = time.time()
            ms = aggregate_max(ev0.elapsed_time(ev1), world, dev)
            total_atoms = aggregate_sum(float(self.n), world, dev)
            n_zbl, n_fp64 = g.nep_zbl_last_counts()
            return {"ms": ms, "ms_per_step": ms / K, "value": total_atoms * K / (ms * 1e-3), "total_atoms": total_atoms,
                    "launches": g.nep_zbl_launch_count() - l0, "rebuilds": g.md_get_counters()[1] - reb0,
                    "forced_rebuilds": forced, "energy_drift_ev_per_atom": (sum(g.md_energies()) - e0) / self.n,
                    "zbl_atoms": n_zbl, "fp64_atoms": n_fp64, "window": (t0, t1),
                    "clocks": sampler.summary(t0, t1) if sampler else None, "graph": g.nep_zbl_uses_graph()}

        def profiled_steps(self, Kp):
            """Per-kernel CUDA-event spans (plain stream launches with events between the kernel groups)."""
            g, w = self.g, self.w
            g.nep_zbl_profile(True)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            g.md_run(Kp, w.dt_max, w.max_displacement)
            b.record(stream)
            prof = g.nep_zbl_profile_read()
            ms_step = a.elapsed_time(b) / Kp
            kern_ms = {k: v[0] / v[1] for k, v in prof.items() if v[1]}
            share = {k: round(v[0] / Kp / ms_step, 4) for k, v in prof.items() if v[1]}
            # one list rebuild: the rebuild slot of a step that rebuilds minus that of a step that does not (the
            # chain is enqueued every step in this mode and exits early unless the flag is set)
            reb = []
            for _ in range(3):
                g.md_request_rebuild()
                g.md_run(1, w.dt_max, w.max_displacement)
                p1 = g.nep_zbl_profile_read()
                g.md_run(1, w.dt_max, w.max_displacement)
                p0 = g.nep_zbl_profile_read()
                reb.append(p1["rebuild"][0] - p0["rebuild"][0])
            g.nep_zbl_profile(False)
            return ms_step, kern_ms, share, float(np.median(reb))

        def close(self):
            self.g.close()
            self.pos = self.vel = self.types = None
            torch.cuda.empty_cache()

    main_run = Run(args.workload, args.cells)
    n, w, g = main_run.n, main_run.w, main_run.g
    dt_max, max_disp = w.dt_max, w.max_displacement
    r = main_run.timed_steps()
    ms, value, total_atoms, clocks = r["ms"], r["value"], r["total_atoms"], r["clocks"]

    # ---- same steps, L2 flushed between steps (per-step event pairs; the flush is outside them)
    flush = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=dev)
    Kf = min(K, args.flush_steps)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(Kf)]
    with torch.cuda.stream(stream):
        for a, b in evs:
            flush.fill_(1)
            a.record(stream)
            g.md_step(dt_max, max_disp)
            b.record(stream)
    barrier()
    ms_flushed = aggregate_max(sum(a.elapsed_time(b) for a, b in evs) / Kf, world, dev)
    del flush

    ms_prof_step, kern_ms, kern_share, rebuild_ms = main_run.profiled_steps(min(K, 200))
    ffma_measured = g.nep_zbl_ffma_peak()

    # ---- end to end through the C ABI with HOST buffers (md_step_host): H2D + step + D2H per step
    hp = torch.from_numpy(w.pos.copy()).pin_memory()
    hv = torch.from_numpy(w.vel.copy()).pin_memory()
    main_run.fresh_state()
    Ke = min(K, args.e2e_steps)
    for _ in range(min(W, 5)):
        g.md_step_host(hp, hv, dt_max, max_disp)
    eve0, eve1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.perf_counter()
    eve0.record(stream)
    for _ in range(Ke):
        g.md_step_host(hp, hv, dt_max, max_disp)
    eve1.record(stream)
    barrier()
    wall_e2e = (time.perf_counter() - t0) * 1e3
    ms_e2e = aggregate_max(max(eve0.elapsed_time(eve1), wall_e2e), world, dev)
    e2e_value = total_atoms * Ke / (ms_e2e * 1e-3)
    del hp, hv

    # ---- SURVEY 8(f) NEXT rows, same workload: border-layer Nose-Hoover chain and Wigner-Seitz count
    next_rows = None
    hbm_peak_ = 6650.0
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        hbm_peak_ = float(peaks.get("hbm_gbs", 6650.0))
    except OSError:
        pass
    if world == 1 and not args.no_next:
        from paper_2305_08140_b200 import workloads as wl_
        group = torch.from_numpy(wl_.border_group(w.pos, w.box, w.pbc)).to(dev)
        main_run.fresh_state()
        pos = main_run.pos
        g.md_set_thermostat(group, 300.0, 100.0, 4)
        Kn = min(K, 200)
        g.md_run(W, dt_max, max_disp)
        evn0, evn1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        evn0.record(stream)
        g.md_run(Kn, dt_max, max_disp)
        evn1.record(stream)
        barrier()
        ms_nhc = evn0.elapsed_time(evn1) / Kn
        t_group = g.md_get_thermostat()[2]
        g.md_set_thermostat(None, 300.0, 100.0, 4)
        site = torch.from_numpy(w.pos.copy()).to(dev)       # reference = the initial lattice
        g.wigner_seitz_set_reference(site, w.box, w.pbc)
        for _ in range(3):
            g.wigner_seitz_count(pos, want_nearest=True, want_occupancy=True)
        evw0, evw1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 20
        barrier()
        evw0.record(stream)
        for _ in range(reps):
            _, _, ws_counts = g.wigner_seitz_count(pos, want_nearest=True, want_occupancy=True)
        evw1.record(stream)
        barrier()
        ms_ws = evw0.elapsed_time(evw1) / reps
        ws_gbs = WS_BYTES_PER_ATOM * n / (ms_ws * 1e-3) / 1e9
        next_rows = {
            "nhc_border_layer": {"ms_per_step": ms_nhc, "atom_steps_per_s": n / (ms_nhc * 1e-3), "steps": Kn,
                                 "group_atoms": int(group.sum().item()), "t_group_K": t_group,
                                 "chain": 4, "tau_fs": 100.0},
            "wigner_seitz": {"ms_per_count": ms_ws, "atoms_per_s": n / (ms_ws * 1e-3), "sites": n,
                             "vacancies": ws_counts[0], "interstitials": ws_counts[1],
                             "roofline": {"bound": "hbm", "achieved": ws_gbs, "peak": hbm_peak_, "unit": "GB/s",
                                          "frac": ws_gbs / hbm_peak_, "bytes_per_atom": WS_BYTES_PER_ATOM},
                             "includes": "occupancy memset, assignment, count, 16-byte D2H of the totals, stream sync"},
        }
        del site, group
    props = torch.cuda.get_device_properties(dev)
    workspace_bytes = g.workspace_bytes
    main_run_mode = g.nep_zbl_network_mode()
    main_run.close()

    # ---- the other configs of BASELINE.json in the same run (device-resident timing only)
    per_config = None
    if world == 1 and args.per_config and args.cells is None:
        per_config = {}
        for name in [c for c in ("config2", "config3", "config5") if c != args.workload]:
            run = Run(name)
            rr = run.timed_steps()
            _, kms, _, reb_ms = run.profiled_steps(min(K, 50))
            per_config[name] = {"atoms": run.n, "ms_per_step": rr["ms_per_step"], "value": rr["value"], "steps": K,
                                "list_rebuilds_in_timed_region": int(rr["rebuilds"]),
                                "forced_rebuilds": rr["forced_rebuilds"], "rebuild_ms": reb_ms,
                                "kernel_ms": {k: round(v, 5) for k, v in kms.items()},
                                "zbl_atoms": rr["zbl_atoms"], "fp64_atoms": rr["fp64_atoms"],
                                "energy_drift_ev_per_atom": rr["energy_drift_ev_per_atom"],
                                "workspace_gib": run.g.workspace_bytes / 2 ** 30, "clocks": rr["clocks"]}
            run.close()
    if sampler:
        sampler.stop()

    if rank != 0:
        return 0

    # ---- roofline of the dominant kernel
    force_kernels = {k: kern_ms[k] for k in ("k_radial", "k_angular_nn", "k_force") if k in kern_ms}
    dom = max(force_kernels, key=force_kernels.get)
    sm_max_mhz = float(peaks.get("sm_max_mhz", (clocks or {}).get("sm_max_mhz") or 1965.0))
    alu_peak = props.multi_processor_count * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12     # TFLOP/s
    flop_table = PAPER_FLOP_PER_ATOM if args.workload == "paper" else FLOP_PER_ATOM
    achieved = flop_table[dom] * n / (kern_ms[dom] * 1e-3) / 1e12
    hbm_peak = hbm_peak_
    traffic, traffic_note = (args.traffic_bytes, "--traffic-bytes") if args.traffic_bytes is not None else \
        ncu_traffic(args.workload, dom, args.cells)
    # which kernel the slot "k_angular_nn" timed: the network layer runs on the tensor cores in k_angular_tc
    # (nep_zbl_network_mode 3); its S6 flops are then tensor-pipe work (3 tf32 products per fp32 product), the
    # rest of the kernel CUDA-core work -- `achieved` counts the algorithmic flops of the whole kernel either way
    nn_mode = main_run_mode
    step_flop = PAPER_STEP_FLOP if args.workload == "paper" else STEP_FLOP
    network = {"mode": nn_mode,
               "kernel": {0: "k_angular_nn (FFMA)" if args.workload != "paper" else "k_angular_nn_split (FFMA)",
                          1: "k_angular_nn (mma.sync 3xTF32)", 2: "k_angular_nn (tcgen05, block-synchronous)",
                          3: "k_angular_tc (tcgen05 3xTF32, accumulators in tensor memory, two-tile pipeline)" if args.workload != "paper"
                          else "k_angular_split_tc (tcgen05 3xTF32, four lanes per atom in the passes, one row per thread in the network)"}.get(nn_mode),
               "tensor_core_flop_per_atom": step_flop["S6"] if nn_mode in (1, 2, 3) else 0.0,
               "cuda_core_flop_per_atom": flop_table["k_angular_nn"] - (step_flop["S6"] if nn_mode in (1, 2, 3) else 0.0)}
    if "k_angular_nn" in kern_ms:
        network["cuda_core_tflops"] = network["cuda_core_flop_per_atom"] * n / (kern_ms["k_angular_nn"] * 1e-3) / 1e12
        network["cuda_core_frac_of_alu_peak"] = network["cuda_core_tflops"] / alu_peak
    roofline = {"kernel": dom if not (dom == "k_angular_nn" and nn_mode == 3) else
                ("k_angular_split_tc" if args.workload == "paper" else "k_angular_tc"),
                "bound": "alu", "achieved": achieved, "peak": alu_peak, "unit": "TFLOP/s",
                "frac": achieved / alu_peak, "network": network, "traffic": traffic, "traffic_note": traffic_note,
                "peak_source": f"derived: {props.multi_processor_count} SM x {FP32_LANES_PER_SM} FP32 lanes x 2 x {sm_max_mhz:.0f} MHz",
                "ffma_measured_tflops": ffma_measured, "ms_per_launch": kern_ms[dom],
                "flop_per_atom": flop_table[dom], "units_per_launch": n,
                # every force kernel and the whole step against the same ALU peak (algorithmic flops of DESIGN.md)
                "alu": {k: {"achieved_tflops": flop_table[k] * n / (kern_ms[k] * 1e-3) / 1e12,
                            "frac": flop_table[k] * n / (kern_ms[k] * 1e-3) / 1e12 / alu_peak}
                        for k in flop_table if k in kern_ms},
                "step": {"flop_per_atom": sum(flop_table.values()),
                         "achieved_tflops": sum(flop_table.values()) * n / (ms / K * 1e-3) / 1e12,
                         "frac": sum(flop_table.values()) * n / (ms / K * 1e-3) / 1e12 / alu_peak},
                "hbm": {k: {"achieved_gbs": BYTES_PER_ATOM[k] * n / (kern_ms[k] * 1e-3) / 1e9,
                            "frac": BYTES_PER_ATOM[k] * n / (kern_ms[k] * 1e-3) / 1e9 / hbm_peak}
                        for k in BYTES_PER_ATOM if k in kern_ms},
                "hbm_peak_gbs": hbm_peak, "hbm_peak_source": "measured" if peaks else "fallback"}

    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        cpu_baseline, _ = oracle_md_rate(args.workload, None, 0, budget_s=12.0)
        cpu_baseline["single_evaluations"] = oracle_single_evaluations()

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": args.workload, "atoms_per_gpu": n, "dt_max_fs": dt_max,
                   "max_displacement_A": (None if not np.isfinite(max_disp) else max_disp), "skin_A": w.model["skin"],
                   "model": MODEL_DESC.get(args.workload, DEFAULT_MODEL_DESC),
                   "precision": "fp32 descriptors/network/forces (fp64 re-evaluation of disordered sites), "
                                "fp64 positions/velocities/ZBL/energy sums",
                   "parallelism": "single GPU" if world == 1 else f"{world} independent replicas",
                   "l2": f"no flush for `value` (consecutive steps of one trajectory; workspace {workspace_bytes / 2**20:.0f} MiB "
                         f"> {L2_BYTES / 2**20:.0f} MiB L2); `ms_per_step_l2_flushed` flushes L2 (2x L2 write) before every step",
                   "list_rebuilds_in_timed_region": int(r["rebuilds"]), "forced_rebuilds": r["forced_rebuilds"],
                   "cuda_graph": bool(r["graph"])},
        "ms_per_step_l2_flushed": ms_flushed, "value_l2_flushed": total_atoms / (ms_flushed * 1e-3),
        "ms_per_step_profiled": ms_prof_step, "rebuild_ms": rebuild_ms,
        "kernel_ms": {k: round(v, 5) for k, v in kern_ms.items()}, "kernel_share": kern_share,
        "energy_drift_ev_per_atom": r["energy_drift_ev_per_atom"],
        "zbl_atoms": r["zbl_atoms"], "fp64_atoms": r["fp64_atoms"],
        "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu_baseline,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 48 * n, "d2h_bytes_per_step": 48 * n,
                "steps": Ke, "api": "md_step_host"},
        "gpu_launches": int(r["launches"]),
        "per_config": per_config,
        "next_rows": next_rows,
        "context": {"paper": "1.3e7 atom-step/s, one 40-GB A100, trained W NEP-ZBL (n_max 15/10, 100 neurons), Table IV"},
    }
    print(json.dumps(line))
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="config4",
                    choices=["config2", "config3", "config4", "config5", "alloy", "paper"])
    ap.add_argument("--no-per-config", dest="per_config", action="store_false",
                    help="skip the other BASELINE.json configs (config2/3/5) timed in the same run")
    ap.add_argument("--cells", type=int, default=None, help="override the cell count (debug only)")
    ap.add_argument("--e2e-steps", type=int, default=200)
    ap.add_argument("--flush-steps", type=int, default=100)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-next", action="store_true", help="skip the SURVEY 8(f) NEXT rows (thermostat, Wigner-Seitz)")
    ap.add_argument("--traffic-bytes", type=float, default=None,
                    help="dram bytes per launch of the dominant kernel from the committed ncu capture")
    args = ap.parse_args(argv)
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())

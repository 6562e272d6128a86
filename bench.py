#!/usr/bin/env python
"""bench.py -- effective HBM GB/s per SLDG substep and per Strang step (fp64) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c4|c4o3|c3|c0|paper|c1o2|c1o3|c2]

A "step" is one Strang step z(dt/2) v(dt/2) xy(dt) v(dt/2) z(dt/2) over the whole 4d array (all rows of
SURVEY.md 8(a)).  Metric (BASELINE.json / PAPER.md:380): 2*|f|*8 bytes per substep, 10*|f|*8 bytes per
Strang step, divided by device time -- ALGORITHMIC (unfused-equivalent) bytes: the fused step physically makes three
passes over f, so `value` can exceed the copy rate; `hbm_gbs_actual` beside it is bytes really moved / time.
One JSON line on stdout (rank 0).  The default workload is BASELINE.json configs[4]; its o = 3 half
(96x96x48x48 cells) is timed in the same run and reported as the sub-record "o3", the paper's own grid (64x64x64x128 cells,
o = 2) as the sub-record "paper_grid".

N > 1 (torchrun): the path does not shard (north_star: one GPU, no collectives) -> N independent
replicas, one per GPU; value = sum over replicas / max-over-ranks time.  "scaling": "weak".

--impl reference: the CPU oracle (oracle/), as it stands, timed on this box's host cores on a bounded
sample of the same workload.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2212_03036_b200 import inputs  # noqa: E402

WORKLOADS = {
    # name: (nx, ny, nz, nv, order, dt, description)
    "c4": (128, 128, 64, 64, 2, 4.0, "BASELINE.json configs[4]: large 4d ITG, 128x128x64x64 cells, o=2, dt=4"),
    "c4o3": (96, 96, 48, 48, 3, 4.0, "BASELINE.json configs[4] (o=3 variant): 96x96x48x48 cells, o=3, dt=4"),
    "c3": (64, 64, 32, 64, 2, 4.0, "BASELINE.json configs[3]: mid 4d ITG, 64x64x32x64 cells, o=2, dt=4"),
    "c0": (16, 16, 8, 16, 2, 2.0, "BASELINE.json configs[0]: tiny 4d ITG, 16x16x8x16 cells, o=2, dt=2"),
    "paper": (64, 64, 64, 128, 2, 4.0, "the paper's grid 64x64x64x128 cells, o=2 (PAPER.md:348, :431)"),
}
# bounded CPU sample of the same ITG workload (same box, profiles, dt): 1/64 of c4's cells
CPU_SAMPLE = (64, 64, 8, 32)
NOMINAL_PEAK_GBS = 8000.0
CSRC = os.path.join(ROOT, "paper_2212_03036_b200", "csrc")

# Algorithmic fp64 flops of the 2d geometry (DESIGN.md 6.1 derives them from eq. (14)-(18) as implemented: tracing of
# 4 corners + o^2 nodes through the bilinear field, o^2 x o^2 Gauss-Jordan, per non-empty piece the Green's-theorem
# moments over the 4 clipped edges with a (2o-1)-point rule and the contraction to o^4 weights): per target cell and
# per non-empty (target, source) piece.  The 2d apply does 2 o^4 flops per piece and v node (eq. 17).
GEOM_FLOPS = {1: {"cell": 300, "piece": 150}, 2: {"cell": 580, "piece": 830}, 3: {"cell": 2225, "piece": 4700}}


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def source_hash(files):
    """First 16 hex digits of the sha256 over the named csrc files: ties an ncu capture to the kernel source it saw."""
    h = hashlib.sha256()
    for name in files:
        with open(os.path.join(CSRC, name), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_traffic(kernel, workload):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full capture
    (profiles/r02_ncu_traffic.csv: workload,kernel,read_bytes,write_bytes,source files,source sha256/16,capture).
    A row whose kernel sources have changed since the capture is REFUSED (returns None): the number printed must
    belong to the kernel that ran.  (DRAM bytes cannot be counted inside an un-profiled run.)"""
    try:
        with open(os.path.join(ROOT, "profiles", "r02_ncu_traffic.csv")) as fh:
            for row in fh:
                p = [x.strip() for x in row.split(",")]
                if len(p) >= 6 and p[0] == workload and p[1] == kernel:
                    if source_hash(p[4].split()) != p[5]:
                        return None
                    return float(p[2]) + float(p[3])
    except OSError:
        pass
    return None


class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons during the timed region."""

    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def wait_first(self, timeout=3.0):
        """nvidia-smi needs a few tenths of a second to print its first line: the timed region (0.1 s) starts after it."""
        t_end = time.time() + timeout
        while self.proc is not None and not self.rows and time.time() < t_end:
            time.sleep(0.01)

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        # samples inside the timed region; nvidia-smi samples every 100 ms, so a 0.1 s region may hold one or none: then
        # the samples right around it (0.3 s) stand in
        rows = ([r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or
                [r for (t, r) in self.rows if t0 - 0.3 <= t <= t1 + 0.3] or [r for (_, r) in self.rows])
        for r in rows:
            p = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(p[0]))
                smax = float(p[1])
                for n, v in zip(names, p[2:6]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax,
                "reasons": sorted(reasons), "samples": len(sm)}


def max_over_ranks(ms, world, device="cuda"):
    """The time every replica-set number is quoted on: the slowest rank's (all ranks get the same value)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t[0])


def replicas_value(nbytes_per_step_per_rank, ms_per_step, world):
    """Whole-job throughput of `world` independent replicas (no sharding, no collectives on the data path):
    bytes of all replicas over the slowest rank's time."""
    return world * gbs(nbytes_per_step_per_rank, ms_per_step)


def gbs(nbytes, ms):
    return nbytes / (ms * 1e-3) / 1e9 if ms > 0 else None


def _omp_set_threads(n):
    """Thread count of the OpenMP runtime the oracle library runs on (the oracle itself is not touched)."""
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except OSError:
        return False


def _cpu_sample():
    nx, ny, nz, nv = CPU_SAMPLE
    spec = inputs.itg_grid(nx, ny, nz, nv, 2)
    dt = 4.0
    f = inputs.itg_initial_f(spec)
    a, b, Ez, _ = inputs.itg_fields(spec, dt, 0.8)
    what = (f"ITG {nx}x{ny}x{nz}x{nv} cells, o=2 ({spec.dofs} DOFs = 1/64 of c4's), same box/profiles/fields, dt=4")
    return spec, dt, f, a, b, Ez, what


def cpu_oracle_time(steps, warmup):
    """Times the oracle's Strang step, as it stands, on all host cores on a bounded sample; returns (GB/s, ms per
    step, cores, sample)."""
    import oracle

    spec, dt, f, a, b, Ez, what = _cpu_sample()
    tmp = np.empty_like(f)
    for _ in range(warmup):
        oracle.strang_step(spec, f, Ez, a, b, dt, 2, 1, tmp=tmp)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle.strang_step(spec, f, Ez, a, b, dt, 2, 1, tmp=tmp)
    el = (time.perf_counter() - t0) / steps
    sample = f"{what}, {steps} Strang step(s) after {warmup} warm-up"
    return 10.0 * spec.dofs * 8 / el / 1e9, el * 1e3, oracle.num_threads(), sample


def cpu_oracle_baseline():
    """SURVEY.md 8(d) "Oracle timing": the oracle as it stands, (i) on all cores and (ii) on a single thread, wall
    clock per substep (best of 3) with the metric's formula (2 |f| 8 B per substep), plus >= 2 whole Strang steps on all
    cores (10 |f| 8 B per step; that is `value`)."""
    import oracle

    spec, dt, f, a, b, Ez, what = _cpu_sample()
    nbytes = spec.dofs * 8.0
    cores = oracle.num_threads()

    def best_of(fn, n=3):
        best = None
        for _ in range(n):
            t0 = time.perf_counter()
            fn()
            el = time.perf_counter() - t0
            best = el if best is None else min(best, el)
        return best

    def substeps():
        tz = best_of(lambda: oracle.advect_z(spec, f, 0.5 * dt))
        tv = best_of(lambda: oracle.advect_v(spec, f, Ez, 0.5 * dt))
        txy = best_of(lambda: oracle.advect_xy(spec, f, a, b, dt, 2, 1))
        return {"advect_z_gbs": 2 * nbytes / tz / 1e9, "advect_v_gbs": 2 * nbytes / tv / 1e9,
                "advect_xy_gbs": 2 * nbytes / txy / 1e9, "ms": {"z": tz * 1e3, "v": tv * 1e3, "xy": txy * 1e3}}

    all_cores = substeps()
    g = f.copy()
    tmp = np.empty_like(g)
    oracle.strang_step(spec, g, Ez, a, b, dt, 2, 1, tmp=tmp)  # warm-up
    t0 = time.perf_counter()
    for _ in range(2):
        oracle.strang_step(spec, g, Ez, a, b, dt, 2, 1, tmp=tmp)
    step = (time.perf_counter() - t0) / 2
    single = None
    if _omp_set_threads(1):
        single = substeps()
        _omp_set_threads(cores)
    return {"value": 10 * nbytes / step / 1e9, "unit": "GB/s", "cores": cores, "kind": "oracle",
            "sample": f"{what}; 2 Strang steps after 1 warm-up (value); each substep best of 3",
            "ms_per_step": step * 1e3, "substeps_all_cores": all_cores, "substeps_single_thread": single,
            "paper_context": "the paper's tuned OpenMP code: ~23 GB/s on 2x16 cores (PAPER.md:414)"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    steps = max(1, args.steps)
    v, ms, cores, sample = cpu_oracle_time(steps, min(args.warmup, 1))
    line = {
        "impl": "reference", "metric": "effective_hbm_gbs_per_strang_step", "value": v, "unit": "GB/s",
        "n_gpus": args.gpus, "steps": steps, "warmup": min(args.warmup, 1), "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOADS[args.workload][6], "sample": sample},
        "cpu_baseline": {"value": v, "unit": "GB/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def run_xy_only(args):
    """BASELINE.json configs[1]: the 2d step alone on 256x256 cells, batched over 4096 planes that share one velocity
    field; solid-body rotation, one period in 40 steps (trace order 2).  A step = one sldg_advect_xy."""
    import math

    import torch

    from paper_2212_03036_b200.binding import Sldg

    order = 3 if args.workload.endswith("o3") else 2
    spec = inputs.bumps_grid(256, 4096, order)
    s = Sldg(spec)
    s.import_state_host(inputs.bumps_initial_f(spec, seed=1))
    a, b = inputs.rotation_velocity(spec)
    s.set_vxy(torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda(), 0)
    tau = 2.0 * math.pi / 40
    mass0 = float(s.mass().cpu()[0])
    for _ in range(args.warmup):
        s.advect_xy(tau, 2)
    s.check()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record()
    for _ in range(args.steps):
        s.advect_xy(tau, 2)
    ev1.record()
    torch.cuda.synchronize()
    s.check()
    ms = ev0.elapsed_time(ev1) / args.steps
    geom_ms = s.last_timing_ms()[2]
    mass1 = float(s.mass().cpu()[0])
    nbytes = spec.dofs * 8.0
    peak, peak_src = measured_peak()
    v = gbs(2 * nbytes, ms)
    print(json.dumps({
        "metric": "effective_hbm_gbs_per_xy_substep", "value": v, "unit": "GB/s", "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[1]: 2d SLDG alone, 256x256 cells, o={order}, 4096 planes of seeded "
                               "Gaussian bumps, solid-body rotation (one period = 40 steps)", "dofs": spec.dofs,
                   "state_GB": nbytes / 1e9},
        "frac_of_8TBs": v / NOMINAL_PEAK_GBS, "frac_of_measured": v / peak, "xy_geometry_kernel_ms": geom_ms,
        "mass_drift_rel": abs(mass1 - mass0) / abs(mass0), "gpu_launches": int(s.launch_count()),
    }), flush=True)
    s.close()
    return 0


def run_sweeps_only(args):
    """BASELINE.json configs[2]: the 1d sweeps on 128x128x64x64 cells, o=2.  z: per-v-slice Courant numbers up to
    |CFL| = 20; v: E_z a seeded random Fourier field (8 modes per axis, amplitude 0.5) at max |CFL| = 2.5; f = U[0,1] + a
    Maxwellian.  A step = one z sweep + one v sweep (the config's 50 sweeps of each = --steps 50)."""
    import torch

    from paper_2212_03036_b200.binding import Sldg

    spec = inputs.itg_grid(128, 128, 64, 64, 2)
    s = Sldg(spec)
    s.import_state_host(inputs.sweeps_initial_f(spec, seed=3))
    Ez = inputs.fourier_Ez(spec, seed=2)
    s.set_Ez(torch.from_numpy(Ez).cuda())
    dtz, dtv = inputs.sweeps_dt_z(spec, 20.0), inputs.sweeps_dt_v(spec, Ez, 2.5)
    mass0 = float(s.mass().cpu()[0])
    for _ in range(args.warmup):
        s.advect_z(dtz)
        s.advect_v(dtv)
    tz, tv = [], []
    for _ in range(args.steps):
        s.advect_z(dtz)
        tz.append(s.last_timing_ms()[7])
        s.advect_v(dtv)
        tv.append(s.last_timing_ms()[7])
    s.check()
    mass1 = float(s.mass().cpu()[0])
    nbytes = spec.dofs * 8.0
    peak, _ = measured_peak()
    mz, mv = float(np.median(tz)), float(np.median(tv))
    v = gbs(4 * nbytes, mz + mv)
    print(json.dumps({
        "metric": "effective_hbm_gbs_per_sweep", "value": v, "unit": "GB/s", "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": mz + mv, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[2]: 1d sweeps, 128x128x64x64 cells, o=2, z at max |CFL| 20, v with a "
                               "seeded Fourier E_z at max |CFL| 2.5", "dofs": spec.dofs, "state_GB": nbytes / 1e9},
        "advect_z_ms": mz, "advect_z_gbs": gbs(2 * nbytes, mz), "advect_z_frac_of_8TBs": gbs(2 * nbytes, mz) / NOMINAL_PEAK_GBS,
        "advect_v_ms": mv, "advect_v_gbs": gbs(2 * nbytes, mv), "advect_v_frac_of_8TBs": gbs(2 * nbytes, mv) / NOMINAL_PEAK_GBS,
        "frac_of_measured": v / peak, "mass_drift_rel": abs(mass1 - mass0) / abs(mass0),
        "gpu_launches": int(s.launch_count()),
    }), flush=True)
    s.close()
    return 0


def measure_itg(workload, K, Wm, layout, world, rank, local, barrier, with_e2e, per_step_log=None, clocks=True):
    """One ITG workload through the library: K timed Strang steps (device-resident leg), the per-kernel breakdown from
    the library's own CUDA events, the three substeps through their own calls, the roofline of every kernel, and --
    with_e2e -- the same step driven from pinned host buffers through sldg_strang_step_host."""
    import torch

    from paper_2212_03036_b200.binding import Sldg

    nx, ny, nz, nv, order, dt, desc = WORKLOADS[workload]
    spec = inputs.itg_grid(nx, ny, nz, nv, order)
    s = Sldg(spec, layout=layout)

    # synthetic inputs (seedless analytic ITG profile + prescribed ITG-shaped fields), generated on the host
    f0 = inputs.itg_initial_f(spec)
    a, b, Ez, _ = inputs.itg_fields(spec, dt, 0.8)
    s.import_state_host(f0)
    del f0
    Ez_d, a_d, b_d = (torch.from_numpy(x).cuda() for x in (Ez, a, b))
    s.set_Ez(Ez_d)
    s.set_vxy(a_d, b_d, 1)
    mass0 = float(s.mass().cpu()[0])

    # ---------------- device-resident leg -----------------------------------------------------------
    sampler = ClockSampler(local)
    if rank == 0 and clocks:
        sampler.start()
    for _ in range(Wm):
        s.strang_step(dt)
    s.check()
    if rank == 0 and clocks:
        sampler.wait_first()
    launches0 = s.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_wall0 = time.time()
    ev0.record()
    log = open(per_step_log, "w") if (per_step_log and rank == 0) else None
    for n in range(K):
        s.strang_step(dt)
        if log:
            t = s.last_timing_ms()
            m = float(s.mass().cpu()[0])
            log.write(json.dumps({"step": n, "ms": [float(x) for x in t[:6]], "total_ms": float(t[7]),
                                  "strang_gbs": gbs(10 * spec.dofs * 8.0, t[7]),
                                  "mass_drift_rel": abs(m - mass0) / abs(mass0)}) + "\n")
    ev1.record()
    barrier()
    t_wall1 = time.time()
    if log:
        log.close()
    total_ms = ev0.elapsed_time(ev1)
    hist_timed = s.timing_history(min(K, 64))
    launches = s.launch_count() - launches0
    clk = sampler.stop(t_wall0, t_wall1) if (rank == 0 and clocks) else None
    s.check()
    total_ms = max_over_ranks(total_ms, world)
    mass1 = float(s.mass().cpu()[0])

    # the substeps one by one (the calls of the boundary): z(dt/2), v(dt/2), xy(dt), each 2*|f|*8 bytes -- right after the
    # timed steps, in the same power / clock regime (under the 1 kW cap the SM clock sinks over seconds of sustained load:
    # the ALU-bound 2d geometry measured 0.75 ms fresh and 0.91 ms ten seconds later in the same process)
    single = {"z": [], "v": [], "xy": [], "xy_geometry": []}
    nrep = 5
    for name, call in (("z", lambda: s.advect_z(0.5 * dt)), ("v", lambda: s.advect_v(0.5 * dt)), ("xy", lambda: s.advect_xy(dt, 2))):
        for _ in range(2):
            call()  # warm-up of this kernel sequence; then nrep consecutive calls, each timed by the library's own events
        for _ in range(nrep):
            call()
            t = s.last_timing_ms()
            single[name].append(t[7])
            if name == "xy":
                single["xy_geometry"].append(t[2])
    s.check()
    # breakdown of the Strang step: the per-kernel CUDA-event times of the K TIMED steps themselves, from the library's
    # event history (recorded on the library's stream during the timed region, read here: no synchronisation in the loop)
    per = hist_timed
    med = np.median(np.array(per), axis=0)
    fused_zv, fused_vz = bool(int(med[6]) & 2), bool(int(med[6]) & 4)
    blocks = s.debug_counter(1)  # non-empty (target, source) weight blocks of the last 2d step
    sm = {k: float(np.median(v)) for k, v in single.items()}
    sm_min = {k: float(np.min(v)) for k, v in single.items()}
    rho = s.charge_density()
    torch.cuda.synchronize()
    ev0.record()
    rho = s.charge_density(rho)
    ev1.record()
    torch.cuda.synchronize()
    rho_ms = ev0.elapsed_time(ev1)
    fp64_peak = s.debug_fp64_peak(5)  # TFLOP/s, measured here and now (the roof of the ALU-bound kernels)
    # NEXT rows, outside the Strang step: the source-term substep of the delta-g formulation (one in-place pass over f,
    # PAPER.md:269-279; synthetic equilibrium tables and field derivatives of the right shapes) and the field step
    # (conjugate gradients to 1e-10)
    vv = spec.node_coords(3)
    prof = np.ascontiguousarray(np.repeat((-vv * np.exp(-0.5 * vv * vv))[:, None], spec.N[0], axis=1))
    s.set_equilibrium(torch.from_numpy(prof).cuda(), torch.from_numpy(np.ascontiguousarray(-prof)).cuda())
    s.set_source_fields(Ez_d, Ez_d)
    src_ms = []
    for k in range(6):
        s.source_step(1e-3 if k % 2 == 0 else -1e-3)
        src_ms.append(s.last_timing_ms()[7])
    src_ms = float(np.median(src_ms[1:]))
    n0v, Tev = inputs.itg_vertex_profiles(spec)
    s.set_profiles(torch.from_numpy(n0v).cuda(), torch.from_numpy(Tev).cuda(), 1.0)
    s.field_step(1e-10, 2000)                      # cold: zero initial guess
    field_iters_cold, _ = s.field_info()
    s.advect_z(0.5 * dt)                           # the state moves on by a substep, as between the two field steps of
    s.advect_v(0.5 * dt)                           # Algorithm 1; the solver starts from the previous potential
    torch.cuda.synchronize()
    ev0.record()
    s.field_step(1e-10, 2000)
    ev1.record()
    torch.cuda.synchronize()
    field_ms = ev0.elapsed_time(ev1)
    field_iters, field_relres = s.field_info()
    s.set_Ez(Ez_d)          # the field step overwrote the prescribed fields: put them back for the legs below
    s.set_vxy(a_d, b_d, 1)

    nbytes = spec.dofs * 8.0
    step_ms = total_ms / K
    value = replicas_value(10 * nbytes, step_ms, world)
    peak, peak_src = measured_peak()
    sub = {
        "advect_z_gbs": gbs(2 * nbytes, sm["z"]), "advect_v_gbs": gbs(2 * nbytes, sm["v"]),
        "advect_xy_gbs": gbs(2 * nbytes, sm["xy"]),
        "ms_single_calls": sm, "ms_single_calls_min": sm_min,
        "charge_density_gbs": gbs(nbytes, rho_ms),
        "source_step_ms": src_ms, "source_step_gbs": gbs(2 * nbytes, src_ms),
        "source_step_frac_of_measured_copy": gbs(2 * nbytes, src_ms) / measured_peak()[0],
        "field_step_ms": field_ms, "field_step_cg_iterations_max": field_iters, "field_step_relres_max": field_relres,
        "field_step_cg_iterations_cold_start": field_iters_cold,
        "xy_apply_direct_path_blocks_total": s.debug_counter(0),
        "strang_step_fused_sweep_pairs": {"zv": fused_zv, "vz": fused_vz},
        "strang_step_ms": dict(({"zv_fused": float(med[0])} if fused_zv else {"z": float(med[0]), "v": float(med[1])}),
                               xy=float(med[3]),
                               **({"vz_fused": float(med[4])} if fused_vz else {"v2": float(med[4]), "z2": float(med[5])})),
    }
    for k in ("advect_z_gbs", "advect_v_gbs", "advect_xy_gbs"):
        sub[k.replace("_gbs", "_frac_of_8TBs")] = sub[k] / NOMINAL_PEAK_GBS
        sub[k.replace("_gbs", "_frac_of_measured_copy")] = sub[k] / peak

    # ---- roofline of every kernel of the Strang step (SURVEY.md 8(d) "Roofline per step") -------------------------
    # HBM: achieved = the kernel's own algorithmic bytes (16 B per DOF: every kernel reads f once and writes it once
    # -- a fused pair too, that is its point) / its launch duration, against the measured copy rate.
    # fp64: achieved = algorithmic flops / duration against the fp64 FMA rate measured in this run.  2d apply:
    # 2 o^4 flops per weight block and v node, blocks counted from the geometry's headers; 2d geometry: GEOM_FLOPS.
    ncell_z = nx * ny * spec.N[2]
    o4 = order ** 4
    apply_flops = 2.0 * o4 * blocks * spec.N[3]
    geom_flops = GEOM_FLOPS[order]["cell"] * ncell_z + GEOM_FLOPS[order]["piece"] * float(blocks)
    kern = {"xy_apply": float(med[3] - med[2])}
    kern.update({"fused_zv": float(med[0])} if fused_zv else {"advect_z": float(med[0]), "advect_v": float(med[1])})
    kern.update({"fused_vz": float(med[4])} if fused_vz else {"advect_v_2": float(med[4]), "advect_z_2": float(med[5])})
    allk = {}
    for k, t in kern.items():
        base = k[:-2] if k.endswith("_2") else k
        e = {"bound": "hbm", "achieved": gbs(2 * nbytes, t), "peak": peak, "unit": "GB/s",
             "frac": gbs(2 * nbytes, t) / peak, "launch_ms": t, "share_of_step": t / float(med[7]),
             "algorithmic_bytes_per_launch": 2 * nbytes, "traffic": ncu_traffic(base, workload)}
        if k == "xy_apply":
            tf = apply_flops / (t * 1e-3) / 1e12
            e.update({"hbm_frac": e["frac"], "fp64_tflops": tf, "fp64_frac": tf / fp64_peak,
                      "algorithmic_flops_per_launch": apply_flops, "blocks_per_cell": blocks / ncell_z})
            if tf / fp64_peak > e["frac"]:  # the roof that binds is the one with less head-room
                e.update({"bound": "alu", "achieved": tf, "peak": fp64_peak, "unit": "TFLOP/s", "frac": tf / fp64_peak})
        allk[k] = e
    gtf = geom_flops / (float(med[2]) * 1e-3) / 1e12
    allk["xy_geometry"] = {"bound": "alu", "achieved": gtf, "peak": fp64_peak, "unit": "TFLOP/s", "frac": gtf / fp64_peak,
                           "launch_ms": float(med[2]), "share_of_step": float(med[2] / med[7]),
                           "algorithmic_flops_per_launch": geom_flops,
                           "traffic": ncu_traffic("xy_geometry", workload)}
    dom = max(kern, key=kern.get)
    roofline = dict(allk[dom])
    roofline.update({"kernel": dom, "peak_source": peak_src if roofline["bound"] == "hbm" else
                     "measured in this run (sldg_debug_fp64_peak: independent fp64 FMA chains on every SM)",
                     "fp64_peak_tflops_measured": fp64_peak, "hbm_peak_gbs_measured": peak, "all": allk})
    # bytes really moved per Strang step: the ncu captures where they are valid for this build, else the algorithmic
    # bytes of each kernel (3 passes over f + the weights written by the geometry and read by the apply)
    w_bytes = float(blocks) * (82 if order == 3 else o4) * 8
    moved = 0.0
    for k, e in allk.items():
        alg = 2 * nbytes + (w_bytes if k == "xy_apply" else 0.0) if k != "xy_geometry" else w_bytes
        moved += e["traffic"] if e["traffic"] else alg
    actual = gbs(moved, float(med[7]))

    rec = {
        "value": value, "ms_per_step": step_ms,
        "accounting": "algorithmic (unfused-equivalent) bytes, 10*|f|*8 B per Strang step as in PAPER.md:380/:394; the "
                      "fused step makes 3 passes over f, so this can exceed the copy rate -- see hbm_gbs_actual",
        "effective_frac_of_8TBs": value / world / NOMINAL_PEAK_GBS,
        "hbm_gbs_actual": actual, "hbm_actual_frac_of_measured_copy": actual / peak,
        "hbm_bytes_moved_per_step": moved,
        "config": {"workload": desc, "cells": [nx, ny, nz, nv], "order": order, "dofs": spec.dofs,
                   "state_GB": nbytes / 1e9, "dt": dt, "trace_order": 2,
                   "cache": f"inputs ({nbytes / 1e9:.1f} GB per array) are far larger than the 126 MB L2; no flush needed",
                   "parallelism": "replicas only (no sharding, no collectives)" if world > 1 else "single GPU",
                   "layout": layout},
        "substeps": sub, "roofline": roofline, "gpu_launches": int(launches), "clocks": clk,
        "mass_drift_rel": abs(mass1 - mass0) / abs(mass0),
    }

    # ---------------- end-to-end leg: host buffers through the C-ABI --------------------------------
    if with_e2e:
        Ez_h, a_h, b_h = (torch.from_numpy(x).pin_memory() for x in (Ez, a, b))
        rho_h = torch.empty(Ez.shape, dtype=torch.float64).pin_memory()
        mass_h = torch.empty(1, dtype=torch.float64).pin_memory()
        for _ in range(min(Wm, 3)):
            s.strang_step_host(dt, Ez_h, a_h, b_h, 1, rho_h, mass_h)
        barrier()
        t0 = time.perf_counter()
        for _ in range(K):
            s.strang_step_host(dt, Ez_h, a_h, b_h, 1, rho_h, mass_h)
        barrier()
        e2e_ms = (time.perf_counter() - t0) * 1e3 / K
        e2e_ms = max_over_ranks(e2e_ms, world)
        rec["e2e"] = {"value": replicas_value(10 * nbytes, e2e_ms, world), "unit": "GB/s", "ms_per_step": e2e_ms,
                      "h2d_bytes_per_step": int(Ez_h.numel() * 8 + a_h.numel() * 8 + b_h.numel() * 8),
                      "d2h_bytes_per_step": int(rho_h.numel() * 8 + 8),
                      "what": "sldg_strang_step_host: pinned Ez,a,b -> device, Strang step, rho and mass -> host; "
                              "f stays resident; the copies run on a second stream under the kernels where the data "
                              "dependences allow (Ez and rho in chunks of y rows, the sweep pairs launched per chunk)"}
        s.check()
        del Ez_h, a_h, b_h, rho_h
    s.close()
    del s, Ez_d, a_d, b_d
    torch.cuda.empty_cache()
    return rec


def run_ours(args):
    import torch
    import torch.distributed as dist

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    K, Wm = args.steps, args.warmup
    rec = measure_itg(args.workload, K, Wm, args.layout, world, rank, local, barrier, True, args.per_step_log)
    o3 = None
    if args.workload == "c4" and not args.no_o3:
        # the other half of BASELINE.json configs[4]: "also run at o=3 on 96x96x48x48 cells", same K and W
        o3 = measure_itg("c4o3", K, Wm, args.layout, world, rank, local, barrier, False, None, clocks=False)
    paper = None
    if args.workload == "c4" and not args.no_paper:
        # the paper's own grid (64x64x64x128 cells, 256 KB planes: the z-tiled pair kernel), like for like with its A100 numbers
        paper = measure_itg("paper", K, Wm, args.layout, world, rank, local, barrier, False, None, clocks=False)
    if rank == 0:
        cpu = cpu_oracle_baseline() if (world == 1 and not args.no_cpu_baseline) else None
        line = {
            "metric": "effective_hbm_gbs_per_strang_step", "value": rec.pop("value"), "unit": "GB/s", "n_gpus": world,
            "steps": K, "warmup": Wm, "ms_per_step": rec.pop("ms_per_step"), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        }
        line.update(rec)
        line["cpu_baseline"] = cpu
        if o3 is not None:
            o3["metric"], o3["unit"], o3["steps"], o3["warmup"] = line["metric"], "GB/s", K, Wm
            line["o3"] = o3
        if paper is not None:
            paper["metric"], paper["unit"], paper["steps"], paper["warmup"] = line["metric"], "GB/s", K, Wm
            line["paper_grid"] = paper
        line["paper_context"] = "A100: z 956, v 760, xy 209 GB/s per substep, ~590 GB/s whole step (PAPER.md:408-429)"
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4", choices=sorted(WORKLOADS) + ["c1o2", "c1o3", "c2"])
    ap.add_argument("--per-step-log", default=None,
                    help="write one JSON line per timed Strang step (substep ms, GB/s, mass drift) to this file; the "
                         "step loop then synchronises every step (BASELINE.json configs[3] asks for these records)")
    ap.add_argument("--layout", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-o3", action="store_true", help="skip the o=3 half of configs[4] (sub-record \"o3\")")
    ap.add_argument("--no-paper", action="store_true", help="skip the paper's own grid (sub-record \"paper_grid\")")
    ap.add_argument("--probe", default=None, choices=["fp64"], help="only measure and print the fp64 FMA roof")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    if args.probe == "fp64":
        from paper_2212_03036_b200.binding import Sldg
        t = Sldg(inputs.itg_grid(4, 4, 2, 4, 2))
        print(json.dumps({"probe": "fp64_fma", "tflops": t.debug_fp64_peak(10), "unit": "TFLOP/s"}), flush=True)
        return 0
    if args.workload in ("c1o2", "c1o3"):
        return run_xy_only(args)
    if args.workload == "c2":
        return run_sweeps_only(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())

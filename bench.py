#!/usr/bin/env python
"""bench.py -- effective HBM GB/s per SLDG substep and per Strang step (fp64) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c4|c4o3|c3|c0|paper]

A "step" is one Strang step z(dt/2) v(dt/2) xy(dt) v(dt/2) z(dt/2) over the whole 4d array (all rows of
SURVEY.md 8(a)).  Metric (BASELINE.json / PAPER.md:380): 2*|f|*8 bytes per substep, 10*|f|*8 bytes per
Strang step, divided by device time.  One JSON line on stdout (rank 0).

N > 1 (torchrun): the path does not shard (north_star: one GPU, no collectives) -> N independent
replicas, one per GPU; value = sum over replicas / max-over-ranks time.  "scaling": "weak".

--impl reference: the CPU oracle (oracle/), as it stands, timed on this box's host cores on a bounded
sample of the same workload.
"""
from __future__ import annotations

import argparse
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
# bounded CPU sample of the same ITG workload (same box, profiles, dt): 1/32 of c4's cells
CPU_SAMPLE = (64, 64, 16, 32)
NOMINAL_PEAK_GBS = 8000.0


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_traffic(kernel, workload):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full capture
    (profiles/ncu_traffic.csv: workload,kernel,read_bytes,write_bytes); None if there is no capture."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as fh:
            for row in fh:
                p = [x.strip() for x in row.split(",")]
                if len(p) >= 4 and p[0] == workload and p[1] == kernel:
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

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for (_, r) in self.rows]
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


def cpu_oracle_time(steps, warmup):
    """Times the oracle, as it stands, on a bounded sample; returns (GB/s, ms per step, cores, sample)."""
    import oracle

    nx, ny, nz, nv = CPU_SAMPLE
    spec = inputs.itg_grid(nx, ny, nz, nv, 2)
    dt = 4.0
    f = inputs.itg_initial_f(spec)
    a, b, Ez, _ = inputs.itg_fields(spec, dt, 0.8)
    tmp = np.empty_like(f)
    for _ in range(warmup):
        oracle.strang_step(spec, f, Ez, a, b, dt, 2, 1, tmp=tmp)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle.strang_step(spec, f, Ez, a, b, dt, 2, 1, tmp=tmp)
    el = (time.perf_counter() - t0) / steps
    sample = (f"ITG {nx}x{ny}x{nz}x{nv} cells, o=2 ({spec.dofs} DOFs = 1/32 of c4), same box/profiles/fields, "
              f"dt=4, {steps} Strang step(s) after {warmup} warm-up")
    return 10.0 * spec.dofs * 8 / el / 1e9, el * 1e3, oracle.num_threads(), sample


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


def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_2212_03036_b200.binding import Sldg

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    nx, ny, nz, nv, order, dt, desc = WORKLOADS[args.workload]
    spec = inputs.itg_grid(nx, ny, nz, nv, order)
    K, Wm = args.steps, args.warmup
    s = Sldg(spec, layout=args.layout)

    # synthetic inputs (seedless analytic ITG profile + prescribed ITG-shaped fields), generated on the host
    f0 = inputs.itg_initial_f(spec)
    a, b, Ez, _ = inputs.itg_fields(spec, dt, 0.8)
    s.import_state_host(f0)
    del f0
    Ez_d, a_d, b_d = (torch.from_numpy(x).cuda() for x in (Ez, a, b))
    s.set_Ez(Ez_d)
    s.set_vxy(a_d, b_d, 1)
    mass0 = float(s.mass().cpu()[0])

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---------------- device-resident leg -----------------------------------------------------------
    for _ in range(Wm):
        s.strang_step(dt)
    s.check()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = s.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_wall0 = time.time()
    ev0.record()
    log = open(args.per_step_log, "w") if (args.per_step_log and rank == 0) else None
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
    launches = s.launch_count() - launches0
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    s.check()
    total_ms = max_over_ranks(total_ms, world)
    mass1 = float(s.mass().cpu()[0])

    # breakdown of the Strang step: a few extra steps, device events inside the library (same stream)
    per = []
    for _ in range(max(3, min(K, 10))):
        s.strang_step(dt)
        per.append(s.last_timing_ms())
    med = np.median(np.array(per), axis=0)
    fused_zv, fused_vz = bool(int(med[6]) & 2), bool(int(med[6]) & 4)
    # the substeps one by one (the calls of the boundary): z(dt/2), v(dt/2), xy(dt), each 2*|f|*8 bytes
    single = {"z": [], "v": [], "xy": [], "xy_geometry": []}
    for _ in range(max(3, min(K, 5))):
        s.advect_z(0.5 * dt)
        single["z"].append(s.last_timing_ms()[7])
        s.advect_v(0.5 * dt)
        single["v"].append(s.last_timing_ms()[7])
        s.advect_xy(dt, 2)
        t = s.last_timing_ms()
        single["xy"].append(t[7])
        single["xy_geometry"].append(t[2])
        s.advect_v(0.5 * dt)
        s.advect_z(0.5 * dt)
    sm = {k: float(np.median(v)) for k, v in single.items()}
    ev0.record()
    rho = s.charge_density()
    ev1.record()
    torch.cuda.synchronize()
    ev0.record()
    rho = s.charge_density(rho)
    ev1.record()
    torch.cuda.synchronize()
    rho_ms = ev0.elapsed_time(ev1)

    nbytes = spec.dofs * 8.0
    step_ms = total_ms / K
    value = replicas_value(10 * nbytes, step_ms, world)
    peak, peak_src = measured_peak()
    sub = {
        "advect_z_gbs": gbs(2 * nbytes, sm["z"]), "advect_v_gbs": gbs(2 * nbytes, sm["v"]),
        "advect_xy_gbs": gbs(2 * nbytes, sm["xy"]),
        "ms_single_calls": sm,
        "charge_density_gbs": gbs(nbytes, rho_ms),
        "xy_apply_direct_path_blocks_total": s.debug_counter(0),
        "strang_step_fused_sweep_pairs": {"zv": fused_zv, "vz": fused_vz},
        "strang_step_ms": dict(({"zv_fused": float(med[0])} if fused_zv else {"z": float(med[0]), "v": float(med[1])}),
                               xy=float(med[3]),
                               **({"vz_fused": float(med[4])} if fused_vz else {"v2": float(med[4]), "z2": float(med[5])})),
    }
    for k in ("advect_z_gbs", "advect_v_gbs", "advect_xy_gbs"):
        sub[k.replace("_gbs", "_frac_of_8TBs")] = sub[k] / NOMINAL_PEAK_GBS
    # Roofline per kernel of the Strang step: achieved = the kernel's own algorithmic bytes (16 B per DOF: every
    # kernel reads f once and writes it once -- a fused pair too, that is its point) / its launch duration.
    kern = {"xy_apply": float(med[3] - med[2])}
    kern.update({"fused_zv": float(med[0])} if fused_zv else {"advect_z": float(med[0]), "advect_v": float(med[1])})
    kern.update({"fused_vz": float(med[4])} if fused_vz else {"advect_v": float(med[4]), "advect_z": float(med[5])})
    dom = max(kern, key=kern.get)
    allk = {k: {"achieved": gbs(2 * nbytes, t), "frac": gbs(2 * nbytes, t) / peak, "launch_ms": t,
                "share_of_step": t / float(med[7]), "traffic": ncu_traffic(k, args.workload)} for k, t in kern.items()}
    allk["xy_geometry"] = {"launch_ms": float(med[2]), "share_of_step": float(med[2] / med[7]), "bound": "alu",
                           "traffic": ncu_traffic("xy_geometry", args.workload)}
    roofline = {"kernel": dom, "bound": "hbm", "achieved": allk[dom]["achieved"], "peak": peak, "unit": "GB/s",
                "frac": allk[dom]["frac"], "traffic": allk[dom]["traffic"], "peak_source": peak_src,
                "algorithmic_bytes_per_launch": 2 * nbytes, "launch_ms": allk[dom]["launch_ms"],
                "share_of_step": allk[dom]["share_of_step"], "all": allk}

    # ---------------- end-to-end leg: host buffers through the C-ABI --------------------------------
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
    e2e = {"value": replicas_value(10 * nbytes, e2e_ms, world), "unit": "GB/s", "ms_per_step": e2e_ms,
           "h2d_bytes_per_step": int(Ez_h.numel() * 8 + a_h.numel() * 8 + b_h.numel() * 8),
           "d2h_bytes_per_step": int(rho_h.numel() * 8 + 8),
           "what": "sldg_strang_step_host: pinned Ez,a,b -> device, Strang step, rho and mass -> host; f stays resident"}
    s.check()

    line = None
    if rank == 0:
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            v, ms, cores, sample = cpu_oracle_time(1, 0)
            cpu = {"value": v, "unit": "GB/s", "cores": cores, "kind": "oracle", "sample": sample,
                   "ms_per_step": ms}
        line = {
            "metric": "effective_hbm_gbs_per_strang_step", "value": value, "unit": "GB/s", "n_gpus": world,
            "steps": K, "warmup": Wm, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": desc, "cells": [nx, ny, nz, nv], "order": order, "dofs": spec.dofs,
                       "state_GB": nbytes / 1e9, "dt": dt, "trace_order": 2,
                       "cache": "inputs (8.6 GB per array at c4) are far larger than the 126 MB L2; no flush needed",
                       "parallelism": "replicas only (no sharding, no collectives)" if world > 1 else "single GPU",
                       "layout": args.layout},
            "frac_of_8TBs": value / world / NOMINAL_PEAK_GBS,
            "substeps": sub, "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
            "gpu_launches": int(launches), "clocks": clocks,
            "mass_drift_rel": abs(mass1 - mass0) / abs(mass0),
            "paper_context": "A100: z 956, v 760, xy 209 GB/s per substep, ~590 GB/s whole step (PAPER.md:408-429)",
        }
        print(json.dumps(line), flush=True)
    s.close()
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
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    if args.workload in ("c1o2", "c1o3"):
        return run_xy_only(args)
    if args.workload == "c2":
        return run_sweeps_only(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())

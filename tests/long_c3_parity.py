"""BASELINE.json configs[3] at FULL size against the oracle: 64x64x32x64 cells, o = 2, dt = 4, 200 Strang steps with the
prescribed ITG-shaped fields; relative L-infinity error of the whole state and relative mass drift every 10 steps.

Not collected by pytest (the oracle needs ~5 s per step on 16 cores: ~20 minutes).  Run once per round on the GPU box,

    python tests/long_c3_parity.py [steps] > gpurun_out/c3_parity.txt

and the table goes into profiles/ (VERDICT r01, item 1c).  tests/test_gpu_configs.py holds the same run on a grid the
driver's pytest budget allows."""
import os
import sys
import time

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

import oracle  # noqa: E402
from paper_2212_03036_b200 import inputs  # noqa: E402


def main():
    import torch

    from paper_2212_03036_b200.binding import Sldg

    steps = int(sys.argv[1]) if len(sys.argv) > 1 else 200
    spec = inputs.itg_grid(64, 64, 32, 64, 2)
    dt = 4.0
    f = inputs.itg_initial_f(spec)
    a, b, Ez, _ = inputs.itg_fields(spec, dt, 0.8)
    s = Sldg(spec)
    s.import_state_host(f)
    s.set_Ez(torch.from_numpy(Ez).cuda())
    s.set_vxy(torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda(), 1)
    ref = f.copy()
    tmp = np.empty_like(ref)
    got = np.empty_like(ref)
    m0 = oracle.mass(spec, f)
    print(f"config 3: {spec.n} cells, o=2, {spec.dofs} DOFs, dt={dt}, oracle on {oracle.num_threads()} threads")
    print("| step | rel Linf (GPU vs oracle) | GPU mass drift | oracle mass drift | oracle s/step |")
    print("|---|---|---|---|---|")
    worst = 0.0
    for n in range(1, steps + 1):
        t0 = time.time()
        oracle.strang_step(spec, ref, Ez, a, b, dt, 2, 1, tmp=tmp)
        t1 = time.time() - t0
        s.strang_step(dt)
        if n % 10 == 0 or n == 1 or n == steps:
            s.export_state_host(got)
            err = float(np.abs(got - ref).max() / np.abs(ref).max())
            worst = max(worst, err)
            mg = float(s.mass().cpu()[0])
            print(f"| {n} | {err:.3e} | {abs(mg - m0) / m0:.2e} | {abs(oracle.mass(spec, ref) - m0) / m0:.2e} | {t1:.2f} |",
                  flush=True)
    s.check()
    print(f"worst rel Linf over the run: {worst:.3e} (bar 1e-11)")
    return 0 if worst <= 1e-11 else 1


if __name__ == "__main__":
    sys.exit(main())

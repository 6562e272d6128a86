"""The paper's validation experiment of the 2d SLDG step through the CUDA library.

Swirling deformation (Table 1): the flow of `inputs.paper_swirl_velocity` with T = 1.5 carries a
C^5 cosine bell away and back; meshes 20^2 ... 160^2, dt = 0.5 dx (rounded so that T is a whole number of steps), the
field evaluated at t^{n+1/2} (R8), second-order tracing (eq. 15).  Reported per mesh: the L2 and L-infinity
errors against the initial condition, their orders, and the relative mass error -- the paper observes order ~2.3-2.4
in L2 and a mass error at machine precision for k = 1.  The time stepper is a callable so that the same study runs on
the CPU oracle in the tests; the default goes through the C-ABI.

    python -m paper_2212_03036_b200.experiments            # prints the table (needs a B200)
"""
from __future__ import annotations

import math

import numpy as np

from . import inputs


def _gpu_stepper(spec, f0):
    import torch

    from .binding import Sldg

    s = Sldg(spec)
    s.import_state(torch.from_numpy(np.ascontiguousarray(f0)).cuda())

    def step(a, b, tau):
        s.set_vxy(torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda(), 1)
        s.advect_xy(tau, 2)

    def finish():
        s.check()
        out = s.export_state().cpu().numpy()
        s.close()
        return out

    return step, finish


def swirl_convergence(meshes=(20, 40, 80, 160), order=2, period=1.5, make_stepper=_gpu_stepper):
    """Rows of Table 1: dicts with mesh, steps, l2, l2_order, linf, linf_order, mass_err."""
    rows = []
    for n in meshes:
        spec = inputs.GridSpec(n=(n, n, 1, 1), order=(order, order, 1, 1), lo=(-math.pi, -math.pi, 0.0, 0.0),
                               hi=(math.pi, math.pi, 1.0, 1.0))
        steps = int(math.ceil(period / (0.5 * spec.h[0]) - 1e-9))
        tau = period / steps
        f0 = inputs.cosine_bell(spec)
        step, finish = make_stepper(spec, f0)
        for k in range(steps):
            a, b = inputs.paper_swirl_velocity(spec, (k + 0.5) * tau, period)
            step(a, b, tau)
        f1 = finish()
        # Gauss-Legendre quadrature of the error at the nodes (weights from the library routine leggauss)
        _, w = np.polynomial.legendre.leggauss(order)
        wx = np.tile(0.5 * w, n) * spec.h[0]
        W = wx[:, None] * wx[None, :]
        d = (f1 - f0)[0, 0]
        row = {"mesh": n, "steps": steps, "l2": float(np.sqrt(np.sum(W * d * d))), "linf": float(np.abs(d).max()),
               "mass_err": float(abs(np.sum(W * f1[0, 0]) - np.sum(W * f0[0, 0])) / np.sum(W * f0[0, 0]))}
        if rows:
            ratio = math.log(n / rows[-1]["mesh"])
            row["l2_order"] = math.log(rows[-1]["l2"] / row["l2"]) / ratio
            row["linf_order"] = math.log(rows[-1]["linf"] / row["linf"]) / ratio
        rows.append(row)
    return rows


def format_table(rows):
    out = ["| mesh | steps | L2 error | L2 order | Linf error | Linf order | mass error |", "|---|---|---|---|---|---|---|"]
    for r in rows:
        out.append(f"| {r['mesh']}x{r['mesh']} | {r['steps']} | {r['l2']:.2e} | {r.get('l2_order', float('nan')):.2f} | "
                   f"{r['linf']:.2e} | {r.get('linf_order', float('nan')):.2f} | {r['mass_err']:.1e} |")
    return "\n".join(out)


if __name__ == "__main__":
    for o in (2, 3):
        print(f"o = {o} (k = {o - 1}); the paper's Table 1 is k = 1: L2 orders 2.39, 2.42, 2.29")
        print(format_table(swirl_convergence(order=o)))

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


def _main_swirl():
    for o in (2, 3):
        print(f"o = {o} (k = {o - 1}); the paper's Table 1 is k = 1: L2 orders 2.39, 2.42, 2.29")
        print(format_table(swirl_convergence(order=o)))


def polar_itg(cells=(64, 64, 32, 64), order=2, dt=4.0, steps=1500, eps=1e-6, every=25):
    """The paper's ion-temperature-gradient run through the library: delta-g formulation in polar
    coordinates, Algorithm 1 with all nine steps, potential from eq. (2).  Returns rows (t, electric energy
    sqrt(int phi^2(r_p, theta, z) dtheta dz), change of the mass of delta-g relative to the total mass int g_eq) every
    `every` steps.  The paper observes an exponential growth of the electric energy until nonlinear saturation."""
    import torch

    from .binding import Sldg

    spec = inputs.polar_grid(*cells, order)
    dg = inputs.polar_initial_dg(spec, eps=eps)
    rv = spec.vertex_coords(0)
    n0, dln_n0, T, _ = inputs.polar_profiles(rv)
    _, dv, dr = inputs.polar_equilibrium(spec)
    cu = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
    s = Sldg(spec)
    s.import_state_host(dg)
    s.set_polar_profiles(cu(rv * n0), cu(dln_n0), cu(T))
    s.set_equilibrium(cu(dv), cu(dr))
    ip = int(round((inputs.POLAR_RP - spec.lo[0]) / spec.h[0]))      # the r vertex at r_p
    w = spec.h[1] * spec.h[2] / spec.order[2]
    geq, _, _ = inputs.polar_equilibrium(spec)
    _, wq = np.polynomial.legendre.leggauss(order)
    wr = np.tile(0.5 * wq, spec.n[0]) * spec.h[0]
    wv = np.tile(0.5 * wq, spec.n[3]) * spec.h[3]
    scale = float((geq * wv[:, None] * wr[None, :]).sum() * (spec.hi[1] - spec.lo[1]) * (spec.hi[2] - spec.lo[2]))  # int g_eq
    m0 = float(s.mass().cpu()[0])
    rows = []
    from .binding import SldgError
    for n in range(steps + 1):
        if n % every == 0:
            try:  # the run ends where an upstream cell leaves the 3x3 stencil: the nonlinear phase
                s.check()
            except SldgError as err:
                rows.append({"t": n * dt, "electric": float("nan"), "mass_change": float("nan"), "stopped": str(err)})
                break
            s.polar_field_step()
            phi = s.get_polar_phi()
            e = float(torch.sqrt((phi[:, :, ip] ** 2).sum() * w))
            rows.append({"t": n * dt, "electric": e, "mass_change": abs(float(s.mass().cpu()[0]) - m0) / scale})
        if n < steps:
            s.step_algorithm1_polar(dt)
    s.close()
    return rows


def growth_rate(rows, t0, t1):
    """Least-squares slope of log(electric energy) over t in [t0, t1]."""
    sel = [(r["t"], math.log(r["electric"])) for r in rows if t0 <= r["t"] <= t1 and r["electric"] > 0]
    t = np.array([a for a, _ in sel])
    y = np.array([b for _, b in sel])
    return float(np.polyfit(t, y, 1)[0])


if __name__ == "__main__":
    import sys

    if len(sys.argv) > 1 and sys.argv[1] == "itg":
        steps = int(sys.argv[2]) if len(sys.argv) > 2 else 1500
        rows = polar_itg(steps=steps)
        print("| t | electric energy | change of the total mass (relative to int g_eq) |")
        print("|---|---|---|")
        for r in rows:
            print(f"| {r['t']:.0f} | {r['electric']:.4e} | {r['mass_change']:.1e} |" + (f" {r['stopped']}" if "stopped" in r else ""))
        rows = [r for r in rows if "stopped" not in r]
        T = rows[-1]["t"]
        for a, b in ((0.2 * T, 0.5 * T), (0.4 * T, 0.7 * T), (0.5 * T, 0.9 * T)):
            print(f"growth rate of the electric energy over t in [{a:.0f}, {b:.0f}]: {growth_rate(rows, a, b):.5f}")
    else:
        _main_swirl()

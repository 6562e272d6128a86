"""CPU oracle of the delta-g formulation's source term and its time step -- TEST INFRASTRUCTURE.

Plain NumPy, fp64, from PAPER.md:51 (eq. 3), :269-279 (section 3.5) and Algorithm 1.  Axis 0 of the grid
is r, axis 1 theta; the advections are those of oracle/sldg_oracle.c with the drift given at the vertices and the
half-step look-up periodic in theta only (vel_periodic = 2).  Pins: tests/test_oracle_polar.py."""
from __future__ import annotations

import numpy as np


def source_step(f, dz_phi, dth_phi, dv_geq, dr_geq, tau):
    """dg + tau (d_z phi d_v g_eq + d_theta phi d_r(g_eq / r))  -- the update printed at PAPER.md:279.
    f [Nz][Nv][Nth][Nr]; dz_phi, dth_phi [Nz][Nth][Nr]; dv_geq, dr_geq [Nv][Nr]."""
    return f + tau * (dz_phi[:, None, :, :] * dv_geq[None, :, None, :] + dth_phi[:, None, :, :] * dr_geq[None, :, None, :])


def strang_step_sources(spec, f, fields, dv_geq, dr_geq, dt):
    """Algorithm 1 steps 2-4, 6-9 with given fields: source(dt/2), z(dt/2), v(dt/2), 2d(dt) with
    second-order tracing, v(dt/2), z(dt/2), source(dt/2)."""
    import oracle

    f = source_step(f, fields["dz_phi"], fields["dth_phi"], dv_geq, dr_geq, 0.5 * dt)
    f = np.ascontiguousarray(f)
    f = oracle.strang_step(spec, f, fields["Ez"], fields["a"], fields["b"], dt, 2, 2)
    return source_step(f, fields["dz_phi"], fields["dth_phi"], dv_geq, dr_geq, 0.5 * dt)

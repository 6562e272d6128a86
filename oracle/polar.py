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


# ---- the paper's quasi-neutrality solver in polar coordinates (eq. (2), :43, :281-283) -------------------
# Field grid: r vertices i = 0..nr (r_min..r_max), theta vertices j < nth (periodic), Nz equidistant z points inside the
# cells at (m + 1/2) h_z / o_z.  "We can use FFT in the (theta, z) plane.  In addition, we use finite differences in the r
# direction.  Thus, for each degree of freedom in the theta and z direction, a tridiagonal linear system has to be solved."

def _gl01(o):
    t, w = np.polynomial.legendre.leggauss(o)
    return 0.5 * (t + 1.0), 0.5 * w


def _lagrange_at(nodes, x):
    out = np.ones(len(nodes))
    for j in range(len(nodes)):
        for m in range(len(nodes)):
            if m != j:
                out[j] *= (x - nodes[m]) / (nodes[j] - nodes[m])
    return out


def polar_resample(spec, rho):
    """rho [Nz][Nth][Nr] at the GL nodes -> [Nz][nth][nr+1] on the field grid: z inside the cell; at a
    vertex the mean of the adjacent cells' polynomials at that corner -- four cells in the interior, two at r_min and
    r_max (only one cell on the radial side), theta periodic."""
    nr, nth, nz, _ = spec.n
    orr, oth, oz, _ = spec.order
    xr, _ = _gl01(orr)
    xt, _ = _gl01(oth)
    xz, _ = _gl01(oz)
    r = rho.reshape(nz, oz, nth, oth, nr, orr)
    Ez = np.array([_lagrange_at(xz, (m + 0.5) / oz) for m in range(oz)])
    r = np.einsum("mq,zqjbia->zmjbia", Ez, r)
    left = np.einsum("a,zmjbia->zmjbi", _lagrange_at(xr, 0.0), r)    # cell i at vertex i
    right = np.einsum("a,zmjbia->zmjbi", _lagrange_at(xr, 1.0), r)   # cell i at vertex i+1
    vr = np.empty(left.shape[:4] + (nr + 1,))
    vr[..., 0] = left[..., 0]
    vr[..., nr] = right[..., nr - 1]
    vr[..., 1:nr] = 0.5 * (right[..., :-1] + left[..., 1:])
    low = np.einsum("b,zmjbi->zmji", _lagrange_at(xt, 0.0), vr)
    up = np.einsum("b,zmjbi->zmji", _lagrange_at(xt, 1.0), vr)
    v = 0.5 * (np.roll(up, 1, axis=2) + low)
    return v.reshape(nz * oz, nth, nr + 1)


def polar_solve_phi(spec, rhs, dln_n0, Te):
    """phi [Nz][nth][nr+1] of eq. (2):
        -[phi_rr + (1/r + n0'/n0) phi_r + phi_thth / r^2] + (phi - <phi>)/Te = rhs,   <phi> = average over z (R21),
    homogeneous Neumann at r_min, homogeneous Dirichlet at r_max.  FFT in (z, theta) (library routine);
    per mode (kz, m) second-order centred differences in r: a tridiagonal system in phi_0 .. phi_{nr-1}; the ghost value
    of the Neumann condition is phi_{-1} = phi_1.  dln_n0, Te: at the r vertices, length nr + 1."""
    from scipy.linalg import solve_banded

    Nz, nth, nr1 = rhs.shape
    nr = nr1 - 1
    h = spec.h[0]
    rv = spec.vertex_coords(0)
    R = np.fft.fft2(rhs, axes=(0, 1))
    mth = np.fft.fftfreq(nth, 1.0 / nth)              # integer mode numbers of d/dtheta
    P = np.zeros_like(R)
    for kz in range(Nz):
        for j in range(nth):
            ab = np.zeros((3, nr))
            for i in range(nr):
                adv = (1.0 / rv[i] + dln_n0[i]) / (2.0 * h)
                diag = 2.0 / h ** 2 + mth[j] ** 2 / rv[i] ** 2 + (1.0 / Te[i] if kz != 0 else 0.0)
                lo = -1.0 / h ** 2 + adv              # coefficient of phi_{i-1}
                hi = -1.0 / h ** 2 - adv              # coefficient of phi_{i+1}
                if i == 0:
                    hi, lo = hi + lo, 0.0             # phi_{-1} = phi_1
                ab[1, i] = diag
                if i + 1 < nr:
                    ab[0, i + 1] = hi
                if i > 0:
                    ab[2, i - 1] = lo
            sol = solve_banded((1, 1), ab, R[kz, j, :nr])
            P[kz, j, :nr] = sol
    return np.real(np.fft.ifft2(P, axes=(0, 1)))


def polar_derive(spec, phi):
    """Drift and field derivatives on the field grid (second-order differences):
    a = -d_theta phi / r (radial), b = d_r phi / r (angular), e = -d_z phi, dth = d_theta phi; a is exactly zero at r_min
    and r_max; d_r phi: centred inside, zero at r_min (Neumann), one-sided second order at r_max."""
    h, hth = spec.h[0], spec.h[1]
    hz = spec.h[2] / spec.order[2]
    rv = spec.vertex_coords(0)
    dth = (np.roll(phi, -1, axis=1) - np.roll(phi, 1, axis=1)) / (2.0 * hth)
    dr = np.empty_like(phi)
    dr[:, :, 1:-1] = (phi[:, :, 2:] - phi[:, :, :-2]) / (2.0 * h)
    dr[:, :, 0] = 0.0
    dr[:, :, -1] = (3.0 * phi[:, :, -1] - 4.0 * phi[:, :, -2] + phi[:, :, -3]) / (2.0 * h)
    a = -dth / rv[None, None, :]
    a[:, :, 0] = 0.0
    a[:, :, -1] = 0.0
    b = dr / rv[None, None, :]
    e = -(np.roll(phi, -1, axis=0) - np.roll(phi, 1, axis=0)) / (2.0 * hz)
    return a, b, e, dth


def _z_to_nodes(spec, F):
    nz, oz = spec.n[2], spec.order[2]
    Nz = nz * oz
    xz, _ = _gl01(oz)
    out = np.empty_like(F)
    for iz in range(nz):
        for q in range(oz):
            s = (iz + xz[q]) * oz - 0.5
            m0 = int(np.floor(s))
            w = s - m0
            out[iz * oz + q] = (1.0 - w) * F[m0 % Nz] + w * F[(m0 + 1) % Nz]
    return out


def _rt_to_nodes(spec, F):
    """[M][nth][nr+1] vertex values (theta periodic) -> [M][Nth][Nr] bilinear inside each cell."""
    nr, nth = spec.n[0], spec.n[1]
    xr, _ = _gl01(spec.order[0])
    xt, _ = _gl01(spec.order[1])
    Fy = np.roll(F, -1, axis=1)
    out = np.empty((F.shape[0], nth, len(xt), nr, len(xr)))
    for q, eta in enumerate(xt):
        for p, xi in enumerate(xr):
            out[:, :, q, :, p] = ((1 - xi) * (1 - eta) * F[:, :, :-1] + xi * (1 - eta) * F[:, :, 1:]
                                  + (1 - xi) * eta * Fy[:, :, :-1] + xi * eta * Fy[:, :, 1:])
    return out.reshape(F.shape[0], nth * len(xt), nr * len(xr))


def polar_field_step(spec, dg, n0, dln_n0, Te):
    """Algorithm 1 step 1 / 5 in the delta-g formulation: rhs = (1/(r n0)) int dg dv on the field grid,
    potential, drift at the vertices per GL z node (theta wrap row copied), E_z, d_z phi, d_theta phi at the nodes."""
    import oracle

    rho = oracle.charge_density(spec, np.ascontiguousarray(dg))
    rv = spec.vertex_coords(0)
    rhs = polar_resample(spec, rho) / (rv * n0)[None, None, :]
    phi = polar_solve_phi(spec, rhs, dln_n0, Te)
    a, b, e, dth = polar_derive(spec, phi)

    def wrap(F):
        out = np.empty((F.shape[0], F.shape[1] + 1, F.shape[2]))
        out[:, :-1] = F
        out[:, -1] = F[:, 0]
        return out

    Ez = _z_to_nodes(spec, _rt_to_nodes(spec, e))
    return {"phi": phi, "a": wrap(_z_to_nodes(spec, a)), "b": wrap(_z_to_nodes(spec, b)), "Ez": Ez, "dz_phi": -Ez,
            "dth_phi": _z_to_nodes(spec, _rt_to_nodes(spec, dth))}


def polar_algorithm1_step(spec, dg, n0, dln_n0, Te, dv_geq, dr_geq, dt):
    """Algorithm 1, all nine steps: 1 field; 2 source(dt/2); 3 z(dt/2); 4 v(dt/2); 5 field from dg*;
    6 2d(dt); 7 v(dt/2); 8 z(dt/2); 9 source(dt/2) -- steps 6-9 with the fields of step 5."""
    import oracle

    fs = polar_field_step(spec, dg, n0, dln_n0, Te)
    dg = source_step(dg, fs["dz_phi"], fs["dth_phi"], dv_geq, dr_geq, 0.5 * dt)
    dg = oracle.advect_z(spec, np.ascontiguousarray(dg), 0.5 * dt)
    dg = oracle.advect_v(spec, dg, fs["Ez"], 0.5 * dt)
    fs = polar_field_step(spec, dg, n0, dln_n0, Te)
    dg = oracle.advect_xy(spec, dg, fs["a"], fs["b"], dt, 2, 2)
    dg = oracle.advect_v(spec, dg, fs["Ez"], 0.5 * dt)
    dg = oracle.advect_z(spec, dg, 0.5 * dt)
    dg = source_step(dg, fs["dz_phi"], fs["dth_phi"], dv_geq, dr_geq, 0.5 * dt)
    return dg, fs


def polar_algorithm2_step(spec, dg, n0, dln_n0, Te, dv_geq, dr_geq, dt):
    """Algorithm 2, all thirteen steps: 1 field phi^n; predictor from dg^n: 2 source(dt/2), 3 z(dt/2),
    4 v(dt/2), 5 2d(dt/2) with first-order tracing (eq. 14) -> dg^{n+1/2}; 6 field phi^{n+1/2}; corrector from dg^n:
    7 source(dt/2), 8 z(dt/2), 9 v(dt/2), 10 2d(dt) with second-order tracing (eq. 15), 11 v(dt/2), 12 z(dt/2),
    13 source(dt/2)."""
    import oracle

    fs = polar_field_step(spec, dg, n0, dln_n0, Te)                                              # 1
    g = source_step(dg, fs["dz_phi"], fs["dth_phi"], dv_geq, dr_geq, 0.5 * dt)                   # 2
    g = oracle.advect_z(spec, np.ascontiguousarray(g), 0.5 * dt)                                 # 3
    g = oracle.advect_v(spec, g, fs["Ez"], 0.5 * dt)                                             # 4
    g = oracle.advect_xy(spec, g, fs["a"], fs["b"], 0.5 * dt, 1, 2)                              # 5
    fs = polar_field_step(spec, g, n0, dln_n0, Te)                                               # 6
    dg = source_step(dg, fs["dz_phi"], fs["dth_phi"], dv_geq, dr_geq, 0.5 * dt)                  # 7
    dg = oracle.advect_z(spec, np.ascontiguousarray(dg), 0.5 * dt)                               # 8
    dg = oracle.advect_v(spec, dg, fs["Ez"], 0.5 * dt)                                           # 9
    dg = oracle.advect_xy(spec, dg, fs["a"], fs["b"], dt, 2, 2)                                  # 10
    dg = oracle.advect_v(spec, dg, fs["Ez"], 0.5 * dt)                                           # 11
    dg = oracle.advect_z(spec, dg, 0.5 * dt)                                                     # 12
    dg = source_step(dg, fs["dz_phi"], fs["dth_phi"], dv_geq, dr_geq, 0.5 * dt)                  # 13
    return dg, fs

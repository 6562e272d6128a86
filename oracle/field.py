"""CPU oracle of the field step -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain NumPy / SciPy, fp64, written from the paper's description of its field solver (eq. (2), :281-283
section 3.6, :93-103 Algorithm 1 steps 1 and 5, :332-346 the invariants) and the readings DESIGN.md R19-R26 take where
BASELINE.json's Cartesian box needs an adaptation.  Shares nothing with paper_2212_03036_b200/csrc: the linear systems
are ASSEMBLED here as sparse matrices and solved by a library direct solver (the CUDA side is matrix-free conjugate
gradients); resampling and interpolation are written with explicit Lagrange polynomials.

Steps (names follow section 3.6):
  resample_rho     rho at the Gauss-Legendre nodes -> the equidistant field grid: in z "inside the cell" (o points per
                   cell at (m + 1/2)/o), in the (x,y) plane "at the cell corners, where the average is taken since the
                   function is discontinuous"
  solve_phi        -(1/n0) div(n0 grad phi) + (phi - <phi>)/Te = rho/n0 - 1 on the periodic vertex grid, second-order
                   finite differences (R20), <phi> = average over z (R21); the z average decouples the problem into one
                   singular system for <phi> (R22) and one system (A + 1/Te) per z point
  derive_fields    a = -d_y phi / B, b = d_x phi / B, E = -d_z phi by second-order centred differences
  to_nodes         "bilinear interpolation" to the Gauss-Legendre nodes; linear in z (R24)
  field_step       the composition: rho -> (a, b at the vertices per z node, E_z and phi at the nodes)
  diagnostics      electric energy on the circle r = r_p, mass, L2 norm, kinetic and potential energy

Pins: tests/test_oracle_field.py (Fourier closed form for constant coefficients, manufactured solution with second-order
convergence, exactness of the resampling for polynomials, residual of the assembled operator against a stencil written
out in the test, decoupling identities of the z average).
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp
import scipy.sparse.linalg as spla


def lagrange_at(nodes, x):
    """l_j(x) for the Lagrange basis on `nodes` (1d array), x scalar -> array of len(nodes)."""
    o = len(nodes)
    out = np.ones(o)
    for j in range(o):
        for m in range(o):
            if m != j:
                out[j] *= (x - nodes[m]) / (nodes[j] - nodes[m])
    return out


def _gl01(o):
    t, w = np.polynomial.legendre.leggauss(o)
    return 0.5 * (t + 1.0), 0.5 * w


def resample_rho(spec, rho):
    """rho [Nz][Ny][Nx] at the GL nodes -> [Nz][ny][nx] on the field grid.

    z: point m = iz*o + m' sits at local coordinate (m' + 1/2)/o of cell iz; the cell's polynomial is evaluated there.
    (x,y): vertex (i,j) takes the mean of the four adjacent cells' polynomials at that corner (periodic)."""
    nx, ny, nz, _ = spec.n
    ox, oy, oz, _ = spec.order
    xz, _ = _gl01(oz)
    xx, _ = _gl01(ox)
    xy, _ = _gl01(oy)
    r = rho.reshape(nz, oz, ny, oy, nx, ox)
    # z: evaluate inside the cell
    Ez = np.array([lagrange_at(xz, (m + 0.5) / oz) for m in range(oz)])      # [m'][q]
    r = np.einsum("mq,zqjbia->zmjbia", Ez, r)
    # x: value at the left (xi = 0) and right (xi = 1) end of every cell
    l0x, l1x = lagrange_at(xx, 0.0), lagrange_at(xx, 1.0)
    l0y, l1y = lagrange_at(xy, 0.0), lagrange_at(xy, 1.0)
    left = np.einsum("a,zmjbia->zmjbi", l0x, r)     # cell i at its left vertex i
    right = np.einsum("a,zmjbia->zmjbi", l1x, r)    # cell i at its right vertex i+1
    # vertex i: right end of cell i-1, left end of cell i
    vx = 0.5 * (np.roll(right, 1, axis=4) + left)   # [z][m][j][b][i]
    low = np.einsum("b,zmjbi->zmji", l0y, vx)
    up = np.einsum("b,zmjbi->zmji", l1y, vx)
    v = 0.5 * (np.roll(up, 1, axis=2) + low)        # [z][m][j][i]
    return v.reshape(nz * oz, ny, nx)


def assemble_A(spec, n0):
    """Sparse matrix of  A phi = -(1/n0) div(n0 grad phi)  on the periodic nx x ny vertex grid (R20): conservative
    second-order differences, the coefficient on a cell face is the mean of the two vertex values."""
    nx, ny = spec.n[0], spec.n[1]
    hx, hy = spec.h[0], spec.h[1]
    N = nx * ny
    rows, cols, vals = [], [], []
    for j in range(ny):
        for i in range(nx):
            k = j * nx + i
            ip, im, jp, jm = (i + 1) % nx, (i - 1) % nx, (j + 1) % ny, (j - 1) % ny
            nE = 0.5 * (n0[j, i] + n0[j, ip])
            nW = 0.5 * (n0[j, i] + n0[j, im])
            nN = 0.5 * (n0[j, i] + n0[jp, i])
            nS = 0.5 * (n0[j, i] + n0[jm, i])
            c = 1.0 / n0[j, i]
            for (kk, v) in ((j * nx + ip, -c * nE / hx ** 2), (j * nx + im, -c * nW / hx ** 2),
                            (jp * nx + i, -c * nN / hy ** 2), (jm * nx + i, -c * nS / hy ** 2),
                            (k, c * ((nE + nW) / hx ** 2 + (nN + nS) / hy ** 2))):
                rows.append(k)
                cols.append(kk)
                vals.append(v)
    return sp.csr_matrix((vals, (rows, cols)), shape=(N, N))  # duplicates (tiny periodic grids) are summed


def solve_phi(spec, rhs, n0, Te):
    """phi [Nz][ny][nx] from rhs = rho~/n0 - 1 [Nz][ny][nx]:  A phi_m + (phi_m - <phi>)/Te = rhs_m,  <phi> = mean_m phi_m.

    The mean over m gives  A <phi> = mean_m rhs  -- singular on the periodic box (constants); the right-hand side is
    made compatible by subtracting the n0-weighted mean c (sum n0 (rbar - c) = 0; c is round-off for a quasi-neutral
    state) from the source, and the solution is the one with zero mean (R22).  Then
    (A + 1/Te) phi_m = rhs_m - c + <phi>/Te for every m, so that mean_m phi_m = <phi> holds exactly."""
    Nz, ny, nx = rhs.shape
    N = nx * ny
    A = assemble_A(spec, n0)
    rbar = rhs.mean(axis=0).reshape(N)
    n0f = n0.reshape(N)
    c = np.dot(n0f, rbar) / n0f.sum()
    # zero-mean solution of the singular system: bordered matrix [[A, 1], [1^T, 0]]
    ones = np.ones((N, 1))
    K = sp.bmat([[A, sp.csr_matrix(ones)], [sp.csr_matrix(ones.T), None]], format="csc")
    sol = spla.spsolve(K, np.concatenate([rbar - c, [0.0]]))
    pbar = sol[:N]
    M = (A + sp.diags(1.0 / Te.reshape(N))).tocsc()
    lu = spla.splu(M)
    phi = np.empty((Nz, ny, nx))
    for m in range(Nz):
        phi[m] = lu.solve(rhs[m].reshape(N) - c + pbar / Te.reshape(N)).reshape(ny, nx)
    return phi, pbar.reshape(ny, nx)


def derive_fields(spec, phi, B=1.0):
    """(a, b, e) on the field grid [Nz][ny][nx]: a = -d_y phi/B, b = d_x phi/B (eq. (1): the poloidal drift), e = -d_z phi,
    periodic second-order centred differences; z spacing h_z / o_z."""
    hx, hy = spec.h[0], spec.h[1]
    hz = spec.h[2] / spec.order[2]
    a = -(np.roll(phi, -1, axis=1) - np.roll(phi, 1, axis=1)) / (2.0 * hy) / B
    b = (np.roll(phi, -1, axis=2) - np.roll(phi, 1, axis=2)) / (2.0 * hx) / B
    e = -(np.roll(phi, -1, axis=0) - np.roll(phi, 1, axis=0)) / (2.0 * hz)
    return a, b, e


def z_to_nodes(spec, F):
    """Field-grid z points -> the GL z nodes, linear interpolation, periodic (R24).  F [Nz][...] -> [Nz][...].
    z node (cell iz, node q) sits at s = (iz + xi_q) o - 1/2 in units of the field grid's index."""
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


def xy_to_nodes(spec, F):
    """Vertex values [M][ny][nx] (periodic) -> the (x,y) GL nodes [M][Ny][Nx] by bilinear interpolation inside each cell
    (PAPER.md:283)."""
    nx, ny = spec.n[0], spec.n[1]
    ox, oy = spec.order[0], spec.order[1]
    xx, _ = _gl01(ox)
    xy, _ = _gl01(oy)
    Fx = np.roll(F, -1, axis=2)           # vertex i+1
    Fy = np.roll(F, -1, axis=1)           # vertex j+1
    Fxy = np.roll(Fx, -1, axis=1)
    out = np.empty((F.shape[0], ny, oy, nx, ox))
    for bq in range(oy):
        for ap in range(ox):
            xi, eta = xx[ap], xy[bq]
            out[:, :, bq, :, ap] = ((1 - xi) * (1 - eta) * F + xi * (1 - eta) * Fx + (1 - xi) * eta * Fy + xi * eta * Fxy)
    return out.reshape(F.shape[0], ny * oy, nx * ox)


def with_wrap(F):
    """[M][ny][nx] periodic vertex values -> [M][ny+1][nx+1] with the wrap row and column copied (bitwise periodic)."""
    M, ny, nx = F.shape
    out = np.empty((M, ny + 1, nx + 1))
    out[:, :ny, :nx] = F
    out[:, ny, :nx] = F[:, 0, :]
    out[:, :, nx] = out[:, :, 0]
    return out


def field_step(spec, rho, n0, Te, B=1.0):
    """Algorithm 1 steps 1 / 5: rho [Nz][Ny][Nx] at the nodes -> dict with
    phi (field grid), a, b [Nz][ny+1][nx+1] at the cell vertices per z node, Ez and phi_nodes [Nz][Ny][Nx]."""
    rt = resample_rho(spec, rho)
    rhs = rt / n0[None, :, :] - 1.0
    phi, pbar = solve_phi(spec, rhs, n0, Te)
    a, b, e = derive_fields(spec, phi, B)
    return {
        "phi": phi, "phibar": pbar,
        "a": with_wrap(z_to_nodes(spec, a)), "b": with_wrap(z_to_nodes(spec, b)),
        "Ez": z_to_nodes(spec, xy_to_nodes(spec, e)),
        "phi_nodes": z_to_nodes(spec, xy_to_nodes(spec, phi)),
    }


def diagnostics(spec, f, phi, phi_nodes, r_p):
    """The quantities of PAPER.md:332-346 for the Cartesian full-f state (Jacobian 1, R0):
    electric energy sqrt(int phi^2(r_p, theta, z) dtheta dz) with phi sampled bilinearly on the circle of radius r_p
    around the box centre at 4 max(nx, ny) angles (R25), mass, L2 norm, kinetic energy int v^2/2 f, potential energy
    int phi f (their sum is the paper's total energy)."""
    nx, ny, nz, nv = spec.n
    Nz = phi.shape[0]
    hx, hy = spec.h[0], spec.h[1]
    # circle
    nth = 4 * max(nx, ny)
    cx, cy = 0.5 * (spec.lo[0] + spec.hi[0]), 0.5 * (spec.lo[1] + spec.hi[1])
    acc = 0.0
    for t in range(nth):
        th = 2.0 * np.pi * (t + 0.5) / nth
        x, y = cx + r_p * np.cos(th), cy + r_p * np.sin(th)
        sx, sy = (x - spec.lo[0]) / hx, (y - spec.lo[1]) / hy
        i0, j0 = int(np.floor(sx)), int(np.floor(sy))
        wx, wy = sx - i0, sy - j0
        i1, j1 = (i0 + 1) % nx, (j0 + 1) % ny
        i0, j0 = i0 % nx, j0 % ny
        val = ((1 - wx) * (1 - wy) * phi[:, j0, i0] + wx * (1 - wy) * phi[:, j0, i1]
               + (1 - wx) * wy * phi[:, j1, i0] + wx * wy * phi[:, j1, i1])
        acc += float(np.sum(val * val))
    electric = np.sqrt(acc * (2.0 * np.pi / nth) * (spec.h[2] / spec.order[2]))
    # Gauss weights of every DOF along each axis
    W = []
    for d in range(4):
        _, w = _gl01(spec.order[d])
        W.append(np.tile(w, spec.n[d]) * spec.h[d])
    wx_, wy_, wz_, wv_ = W
    v = spec.node_coords(3)
    fw = f * wz_[:, None, None, None] * wv_[None, :, None, None] * wy_[None, None, :, None] * wx_[None, None, None, :]
    mass = float(fw.sum())
    l2 = float(np.sqrt((fw * f).sum()))
    kinetic = float((fw * (0.5 * v * v)[None, :, None, None]).sum())
    potential = float((fw * phi_nodes[:, None, :, :]).sum())
    return {"electric": float(electric), "mass": mass, "l2": l2, "kinetic": kinetic, "potential": potential}


def algorithm1_step(spec, f, n0, Te, dt, B=1.0):
    """One step of Algorithm 1 for the Cartesian full-f state (no source terms, R0), in the paper's
    order: 1 field, 3 z(dt/2), 4 v(dt/2), 5 field from the intermediate state, 6 xy(dt) second-order tracing,
    7 v(dt/2), 8 z(dt/2).  Returns the new f and the fields of step 5."""
    import oracle

    fs = field_step(spec, oracle.charge_density(spec, f), n0, Te, B)                # 1
    f = oracle.advect_z(spec, f, 0.5 * dt)                                          # 3
    f = oracle.advect_v(spec, f, fs["Ez"], 0.5 * dt)                                # 4
    fs = field_step(spec, oracle.charge_density(spec, f), n0, Te, B)                # 5
    f = oracle.advect_xy(spec, f, fs["a"], fs["b"], dt, 2, 1)                       # 6
    f = oracle.advect_v(spec, f, fs["Ez"], 0.5 * dt)                                # 7
    f = oracle.advect_z(spec, f, 0.5 * dt)                                          # 8
    return f, fs


def algorithm2_step(spec, f, n0, Te, dt, B=1.0):
    """One step of Algorithm 2, predictor-corrector: 1 field phi^n; predictor 3 z(dt/2), 4 v(dt/2),
    5 xy(dt/2) with first-order tracing (eq. 14) -> f^{n+1/2}; 6 field phi^{n+1/2}; corrector from f^n: 8 z(dt/2),
    9 v(dt/2), 10 xy(dt) with second-order tracing (eq. 15), 11 v(dt/2), 12 z(dt/2)."""
    import oracle

    fs = field_step(spec, oracle.charge_density(spec, f), n0, Te, B)                # 1
    g = oracle.advect_z(spec, f, 0.5 * dt)                                          # 3
    g = oracle.advect_v(spec, g, fs["Ez"], 0.5 * dt)                                # 4
    g = oracle.advect_xy(spec, g, fs["a"], fs["b"], 0.5 * dt, 1, 1)                 # 5
    fs = field_step(spec, oracle.charge_density(spec, g), n0, Te, B)                # 6
    f = oracle.advect_z(spec, f, 0.5 * dt)                                          # 8
    f = oracle.advect_v(spec, f, fs["Ez"], 0.5 * dt)                                # 9
    f = oracle.advect_xy(spec, f, fs["a"], fs["b"], dt, 2, 1)                       # 10
    f = oracle.advect_v(spec, f, fs["Ez"], 0.5 * dt)                                # 11
    f = oracle.advect_z(spec, f, 0.5 * dt)                                          # 12
    return f, fs

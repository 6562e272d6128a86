"""Seeded synthetic inputs for the SLDG hot path (shared by the oracle tests and the CUDA path).

This module holds NONE of the method's arithmetic: no shift matrices, no tracing, no clipping, no
quadrature of the scheme.  It only describes a grid (a plain data container) and samples analytic or
seeded-random functions at the grid's nodes / vertices.  Node positions come from the library routine
``numpy.polynomial.legendre.leggauss`` (the oracle and the CUDA library each carry their own
Gauss-Legendre tables; neither reads this one).

Layouts (canonical):
    f   [Nz][Nv][Ny][Nx]      N. = n. * order.  (DOF index = cell*order + node), fp64
    Ez  [Nz][Ny][Nx]          speed of the v-advection at every (x,y,z) node (eq. 5)
    a,b [Nz][ny+1][nx+1]      poloidal velocity at the cell vertices (eq. 12)

Workloads (recipes, DESIGN.md section "Inputs"; they stand in for the paper's analytic ITG and swirl
set-ups of PAPER.md:297-330, with BASELINE.json's parameters binding):
    itg_*        configs 0, 3, 4  (drift-kinetic ITG profile, Cartesian box)
    bumps_*      config 1         (2d poloidal step alone: rotation and swirl)
    sweeps_*     config 2         (1d sweeps at large Courant numbers)
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np


@dataclasses.dataclass(frozen=True)
class GridSpec:
    """Cells, nodes per cell and box, axis order (x, y, z, v)."""

    n: tuple
    order: tuple
    lo: tuple
    hi: tuple

    def __post_init__(self):
        object.__setattr__(self, "n", tuple(int(c) for c in self.n))
        object.__setattr__(self, "order", tuple(int(c) for c in self.order))
        object.__setattr__(self, "lo", tuple(float(c) for c in self.lo))
        object.__setattr__(self, "hi", tuple(float(c) for c in self.hi))

    @property
    def N(self):
        return tuple(c * o for c, o in zip(self.n, self.order))

    @property
    def h(self):
        return tuple((b - a) / c for a, b, c in zip(self.lo, self.hi, self.n))

    @property
    def dofs(self):
        Nx, Ny, Nz, Nv = self.N
        return Nx * Ny * Nz * Nv

    @property
    def shape(self):
        """Canonical array shape [Nz][Nv][Ny][Nx]."""
        Nx, Ny, Nz, Nv = self.N
        return (Nz, Nv, Ny, Nx)

    def unit_nodes(self, axis):
        """Gauss-Legendre points on (0,1) for this axis (library routine)."""
        t, _ = np.polynomial.legendre.leggauss(self.order[axis])
        return 0.5 * (t + 1.0)

    def node_coords(self, axis):
        """Physical coordinate of every DOF along one axis, length N[axis]."""
        xi = self.unit_nodes(axis)
        cells = np.arange(self.n[axis], dtype=np.float64)
        x = self.lo[axis] + (cells[:, None] + xi[None, :]) * self.h[axis]
        return x.reshape(-1)

    def vertex_coords(self, axis):
        """Physical coordinate of the n+1 cell vertices along one axis."""
        return self.lo[axis] + np.arange(self.n[axis] + 1, dtype=np.float64) * self.h[axis]


# --------------------------------------------------------------------------------------------------
# ITG-shaped workload (configs 0, 3, 4)
# --------------------------------------------------------------------------------------------------

ITG_LZ = 1506.76
ITG_VMAX = 7.32
ITG_BOX = 14.5
ITG_RP = 7.3
ITG_MODE = 15


def itg_grid(nx, ny, nz, nv, order=2):
    return GridSpec(
        n=(nx, ny, nz, nv),
        order=(order, order, order, order),
        lo=(-ITG_BOX, -ITG_BOX, 0.0, -ITG_VMAX),
        hi=(ITG_BOX, ITG_BOX, ITG_LZ, ITG_VMAX),
    )


def _itg_profiles(r):
    t = np.tanh((r - ITG_RP) / 1.45)
    T = np.exp(-0.27586 * 1.45 * t)
    n0 = np.exp(-0.055 * 1.45 * t)
    return T, n0


def itg_initial_f(spec: GridSpec, out=None, eps=1e-6):
    """BASELINE.json configs[0] initial condition sampled at the GL nodes (point values); eps is the
    amplitude of the perturbation (1e-6 in the config; larger values exercise the self-consistent field in tests)."""
    x = spec.node_coords(0)
    y = spec.node_coords(1)
    z = spec.node_coords(2)
    v = spec.node_coords(3)
    X, Y = np.meshgrid(x, y, indexing="xy")  # [Ny][Nx]
    r = np.sqrt(X * X + Y * Y)
    th = np.arctan2(Y, X)
    T, n0 = _itg_profiles(r)
    feq = (n0 / np.sqrt(2.0 * np.pi * T))[None, :, :] * np.exp(-(v * v)[:, None, None] / (2.0 * T)[None, :, :])
    env = eps * np.exp(-((r - ITG_RP) ** 2) / 4.0)  # [Ny][Nx]
    if out is None:
        out = np.empty(spec.shape, dtype=np.float64)
    Lz = spec.hi[2] - spec.lo[2]
    for iz, zz in enumerate(z):
        pert = 1.0 + env * np.cos(ITG_MODE * th + 2.0 * np.pi * zz / Lz)
        np.multiply(feq, pert[None, :, :], out=out[iz])
    return out


def itg_fields(spec: GridSpec, dt, cfl_xy=0.8):
    """Prescribed ITG-shaped potential (SURVEY.md 8(d) note): returns (a, b, Ez, phi0).

    phi = phi0 * exp(-(r-7.3)^2/4) * cos(15 theta + 2 pi z / Lz) on the periodic nx x ny vertex grid per
    z-node; a = -d(phi)/dy, b = d(phi)/dx by centred differences with periodic wrap, the wrap row and
    column copied so that a, b are bitwise periodic; Ez = -d(phi)/dz analytic at the nodes.  phi0 is set
    so that max(|a| dt/hx, |b| dt/hy) = cfl_xy.
    """
    nx, ny, nz, nv = spec.n
    hx, hy, hz, hv = spec.h
    xv = spec.vertex_coords(0)[:-1]
    yv = spec.vertex_coords(1)[:-1]
    z = spec.node_coords(2)
    Lz = spec.hi[2] - spec.lo[2]
    XV, YV = np.meshgrid(xv, yv, indexing="xy")  # [ny][nx]
    rv = np.sqrt(XV * XV + YV * YV)
    thv = np.arctan2(YV, XV)
    envv = np.exp(-((rv - ITG_RP) ** 2) / 4.0)
    phase = ITG_MODE * thv[None, :, :] + (2.0 * np.pi * z / Lz)[:, None, None]
    phi = envv[None, :, :] * np.cos(phase)  # [Nz][ny][nx], unit amplitude
    a_p = -(np.roll(phi, -1, axis=1) - np.roll(phi, 1, axis=1)) / (2.0 * hy)
    b_p = (np.roll(phi, -1, axis=2) - np.roll(phi, 1, axis=2)) / (2.0 * hx)
    peak = max(np.abs(a_p).max() * dt / hx, np.abs(b_p).max() * dt / hy)
    phi0 = cfl_xy / peak
    a = np.empty((phi.shape[0], ny + 1, nx + 1), dtype=np.float64)
    b = np.empty_like(a)
    for dst, src in ((a, a_p), (b, b_p)):
        dst[:, :ny, :nx] = phi0 * src
        dst[:, ny, :nx] = dst[:, 0, :nx]
        dst[:, :, nx] = dst[:, :, 0]
    # Ez = -d(phi)/dz at the (x,y,z) nodes, analytic
    x = spec.node_coords(0)
    y = spec.node_coords(1)
    X, Y = np.meshgrid(x, y, indexing="xy")
    r = np.sqrt(X * X + Y * Y)
    th = np.arctan2(Y, X)
    env = np.exp(-((r - ITG_RP) ** 2) / 4.0)
    ph = ITG_MODE * th[None, :, :] + (2.0 * np.pi * z / Lz)[:, None, None]
    Ez = phi0 * (2.0 * np.pi / Lz) * env[None, :, :] * np.sin(ph)
    return a, b, np.ascontiguousarray(Ez), phi0


def itg_vertex_profiles(spec: GridSpec):
    """n0(r) and T_e(r) = T_i(r) (C_Ti = C_Te, kappa_Ti = kappa_Te) of BASELINE.json configs[0] on the
    periodic nx x ny vertex grid, [ny][nx]: the coefficients of the quasi-neutrality equation (eq. 2)."""
    xv = spec.vertex_coords(0)[:-1]
    yv = spec.vertex_coords(1)[:-1]
    XV, YV = np.meshgrid(xv, yv, indexing="xy")
    T, n0 = _itg_profiles(np.sqrt(XV * XV + YV * YV))
    return np.ascontiguousarray(n0), np.ascontiguousarray(T)


# --------------------------------------------------------------------------------------------------
# 2d-only workload (config 1): batched Gaussian bumps sharing one velocity field
# --------------------------------------------------------------------------------------------------

def bumps_grid(ncell, planes, order):
    return GridSpec(
        n=(ncell, ncell, 1, planes),
        order=(order, order, 1, 1),
        lo=(-math.pi, -math.pi, 0.0, 0.0),
        hi=(math.pi, math.pi, 1.0, 1.0),
    )


def bumps_params(planes, seed=1):
    """Centres c in U[-0.7,0.7]^2 and widths sigma in U[0.10,0.25] per plane."""
    rng = np.random.default_rng(seed)
    c = rng.uniform(-0.7, 0.7, size=(planes, 2))
    sigma = rng.uniform(0.10, 0.25, size=planes)
    return c, sigma


def bumps_initial_f(spec: GridSpec, seed=1, plane_slice=None):
    """One Gaussian bump per v-plane, sampled at the GL nodes; shape [1][planes][Ny][Nx]."""
    c, sigma = bumps_params(spec.n[3], seed)
    if plane_slice is not None:
        c, sigma = c[plane_slice], sigma[plane_slice]
    x = spec.node_coords(0)
    y = spec.node_coords(1)
    dx2 = (x[None, :] - c[:, 0, None]) ** 2  # [P][Nx]
    dy2 = (y[None, :] - c[:, 1, None]) ** 2  # [P][Ny]
    s2 = 2.0 * sigma ** 2
    gx = np.exp(-dx2 / s2[:, None])
    gy = np.exp(-dy2 / s2[:, None])
    f = gy[:, :, None] * gx[:, None, :]
    return np.ascontiguousarray(f[None])


def rotation_velocity(spec: GridSpec):
    """Solid-body rotation u = (-y, x) at the cell vertices; shape [1][ny+1][nx+1] each."""
    xv = spec.vertex_coords(0)
    yv = spec.vertex_coords(1)
    XV, YV = np.meshgrid(xv, yv, indexing="xy")
    return np.ascontiguousarray((-YV)[None]), np.ascontiguousarray(XV[None])


def swirl_velocity(spec: GridSpec, t, period=1.5):
    """u = (sin^2 x sin 2y, -sin^2 y sin 2x) cos(pi t / period) at the cell vertices (config 1)."""
    xv = spec.vertex_coords(0)
    yv = spec.vertex_coords(1)
    XV, YV = np.meshgrid(xv, yv, indexing="xy")
    g = math.cos(math.pi * t / period)
    a = np.sin(XV) ** 2 * np.sin(2.0 * YV) * g
    b = -np.sin(YV) ** 2 * np.sin(2.0 * XV) * g
    # the field is 2 pi periodic: make the wrap row/column bitwise equal
    for u in (a, b):
        u[-1, :] = u[0, :]
        u[:, -1] = u[:, 0]
    return np.ascontiguousarray(a[None]), np.ascontiguousarray(b[None])


# --------------------------------------------------------------------------------------------------
# 1d sweeps workload (config 2)
# --------------------------------------------------------------------------------------------------

def sweeps_initial_f(spec: GridSpec, seed=3):
    """U[0,1] per DOF plus a Maxwellian in v."""
    rng = np.random.default_rng(seed)
    f = rng.random(spec.shape)
    v = spec.node_coords(3)
    f += (np.exp(-0.5 * v * v) / math.sqrt(2.0 * math.pi))[None, :, None, None]
    return f


def sweeps_dt_z(spec: GridSpec, cfl=20.0):
    """dt such that max |v| dt / hz = cfl over the v nodes."""
    v = spec.node_coords(3)
    return cfl * spec.h[2] / np.abs(v).max()


def fourier_Ez(spec: GridSpec, seed=2, modes=8, amplitude=0.5):
    """Seeded smooth random Fourier field, 8 modes per axis, scaled to max |Ez| = amplitude."""
    rng = np.random.default_rng(seed)
    Nx, Ny, Nz, _ = spec.N
    ck = rng.random((modes, modes, modes))
    ph = rng.uniform(0.0, 2.0 * np.pi, size=(modes, modes, modes))
    k = np.arange(modes, dtype=np.float64)
    K2 = k[:, None, None] ** 2 + k[None, :, None] ** 2 + k[None, None, :] ** 2
    ck = ck / (1.0 + K2)
    xt = [(spec.node_coords(ax) - spec.lo[ax]) / (spec.hi[ax] - spec.lo[ax]) for ax in range(3)]
    # S = Re sum_k c_k exp(i(2 pi k.x + phi_k)), evaluated axis by axis
    ex = np.exp(2j * np.pi * k[:, None] * xt[0][None, :])  # [kx][Nx]
    ey = np.exp(2j * np.pi * k[:, None] * xt[1][None, :])  # [ky][Ny]
    ez = np.exp(2j * np.pi * k[:, None] * xt[2][None, :])  # [kz][Nz]
    coef = ck * np.exp(1j * ph)  # [kx][ky][kz]
    t1 = np.einsum("abc,ax->bcx", coef, ex)
    t2 = np.einsum("bcx,by->cyx", t1, ey)
    S = np.einsum("cyx,cz->zyx", t2, ez).real
    S *= amplitude / np.abs(S).max()
    return np.ascontiguousarray(S)


def sweeps_dt_v(spec: GridSpec, Ez, cfl=2.5):
    return cfl * spec.h[3] / np.abs(Ez).max()


# --------------------------------------------------------------------------------------------------
# Swirling-deformation validation of the 2d step (Table 1)
# --------------------------------------------------------------------------------------------------

def paper_swirl_velocity(spec: GridSpec, t, period=1.5):
    """The paper's swirling deformation flow on [-pi,pi]^2 at the cell vertices:
    d_t u - d_x(cos^2(x/2) sin(y) g u) + d_y(sin(x) cos^2(y/2) g u) = 0,  g(t) = pi cos(pi t / T), i.e. the velocity
    (a, b) = (-cos^2(x/2) sin y, sin x cos^2(y/2)) g(t).  Divergence free, no flow through the box boundary, reverses
    at t = T/2 so that the exact solution at t = T is the initial condition."""
    xv = spec.vertex_coords(0)
    yv = spec.vertex_coords(1)
    XV, YV = np.meshgrid(xv, yv, indexing="xy")
    g = math.pi * math.cos(math.pi * t / period)
    a = -np.cos(0.5 * XV) ** 2 * np.sin(YV) * g
    b = np.sin(XV) * np.cos(0.5 * YV) ** 2 * g
    for u in (a, b):  # 2 pi periodic: the wrap row/column bitwise equal
        u[-1, :] = u[0, :]
        u[:, -1] = u[:, 0]
    return np.ascontiguousarray(a[None]), np.ascontiguousarray(b[None])


def cosine_bell(spec: GridSpec, centre=(0.2 * math.pi, 0.3 * math.pi), radius=0.3 * math.pi):
    """A C^5 cosine bell cos^6(pi r / 2R) for r < R (PAPER.md:303 names the regularity; centre and radius are in the
    paper's ref. [2], which is not available: these are this build's choice).  Shape [1][Nv][Ny][Nx], every v plane
    the same bell."""
    x = spec.node_coords(0)
    y = spec.node_coords(1)
    X, Y = np.meshgrid(x, y, indexing="xy")
    r = np.sqrt((X - centre[0]) ** 2 + (Y - centre[1]) ** 2)
    bell = np.where(r < radius, np.cos(0.5 * math.pi * np.minimum(r, radius) / radius) ** 6, 0.0)
    return np.ascontiguousarray(np.broadcast_to(bell[None, None], (1, spec.N[3], spec.N[1], spec.N[0])))


# --------------------------------------------------------------------------------------------------
# Polar delta-g workload: the paper's own ITG set-up.  Axis 0 is r, axis 1 theta.
# --------------------------------------------------------------------------------------------------

POLAR_RMIN, POLAR_RMAX = 0.1, 14.5
POLAR_LZ = 1506.759067
POLAR_RP = 0.5 * (POLAR_RMAX + POLAR_RMIN)
POLAR_DR = 8.0          # delta r = 4 delta r_n0 / delta r_Ti
POLAR_M, POLAR_N = 5, 1


def polar_grid(nr, nth, nz, nv, order=2, vmax=ITG_VMAX):
    return GridSpec(n=(nr, nth, nz, nv), order=(order, order, order, order),
                    lo=(POLAR_RMIN, 0.0, 0.0, -vmax), hi=(POLAR_RMAX, 2.0 * math.pi, POLAR_LZ, vmax))


def _polar_profile(r, kappa, delta):
    """exp(-kappa delta tanh((r - r_p)/delta)) and its logarithmic derivative -kappa sech^2((r - r_p)/delta)."""
    t = np.tanh((r - POLAR_RP) / delta)
    return np.exp(-kappa * delta * t), -kappa * (1.0 - t * t)


def polar_profiles(r):
    """n0, T_i (= T_e) and their logarithmic derivatives at radii r."""
    rr = np.linspace(POLAR_RMIN, POLAR_RMAX, 20001)
    shape, _ = _polar_profile(rr, 0.055, 2.9)
    integral = float(np.sum(0.5 * (shape[1:] + shape[:-1]) * np.diff(rr)))
    c_n0 = (POLAR_RMAX - POLAR_RMIN) / integral
    n0, dln_n0 = _polar_profile(r, 0.055, 2.9)
    T, dln_T = _polar_profile(r, 0.27586, 1.45)
    return c_n0 * n0, dln_n0, T, dln_T


def polar_equilibrium(spec: GridSpec):
    """g_eq = r f_eq, d_v g_eq and d_r(g_eq / r) = d_r f_eq at the (v, r) nodes, each [Nv][Nr]."""
    r = spec.node_coords(0)[None, :]
    v = spec.node_coords(3)[:, None]
    n0, dln_n0, T, dln_T = polar_profiles(r)
    feq = n0 / np.sqrt(2.0 * np.pi * T) * np.exp(-v * v / (2.0 * T))
    geq = r * feq
    dv_geq = -(v / T) * geq
    dr_feq = feq * (dln_n0 - 0.5 * dln_T + v * v / (2.0 * T) * dln_T)
    return np.ascontiguousarray(geq), np.ascontiguousarray(dv_geq), np.ascontiguousarray(dr_feq)


def polar_initial_dg(spec: GridSpec, eps=1e-6):
    """delta g(t=0) = r f_eq eps exp(-(r - r_p)^2 / delta r) cos(2 pi n z / L + m theta), [Nz][Nv][Ntheta][Nr]."""
    geq, _, _ = polar_equilibrium(spec)
    r = spec.node_coords(0)
    th = spec.node_coords(1)
    z = spec.node_coords(2)
    env = eps * np.exp(-((r - POLAR_RP) ** 2) / POLAR_DR)
    phase = (2.0 * np.pi * POLAR_N * z / POLAR_LZ)[:, None, None] + POLAR_M * th[None, :, None]
    return np.ascontiguousarray(geq[None, :, None, :] * (env[None, None, :] * np.cos(phase))[:, None, :, :])


def polar_fields(spec: GridSpec, dt, cfl=0.8):
    """Prescribed ITG-shaped potential phi = phi0 w(r) cos(m theta + 2 pi n z / L), w = exp(-(r - r_p)^2 / delta r)
    sin^2(pi (r - r_min)/(r_max - r_min)) (decays to zero at both radial ends, as the paper's phi does).
    Returns a dict: a = -d_theta phi / r, b = d_r phi / r at the vertices [Nz][ntheta+1][nr+1] by centred differences of the
    vertex values (one-sided at the radial ends; a set to exactly zero there; the theta wrap row copied), Ez
    = -d_z phi analytic at the nodes, dz_phi = -Ez, dth_phi = the centred theta difference at the vertices interpolated
    bilinearly to the nodes (its Gauss sum over theta telescopes to zero, the property section 3.5 asks
    for), phi0 such that max(|a| dt / h_r, |b| dt / h_theta) = cfl."""
    nr, nth, nz, nv = spec.n
    hr, hth = spec.h[0], spec.h[1]
    rv = spec.vertex_coords(0)
    thv = spec.vertex_coords(1)[:-1]
    z = spec.node_coords(2)

    def w(r):
        return np.exp(-((r - POLAR_RP) ** 2) / POLAR_DR) * np.sin(np.pi * (r - POLAR_RMIN) / (POLAR_RMAX - POLAR_RMIN)) ** 2

    kz = 2.0 * np.pi * POLAR_N / POLAR_LZ
    phase = POLAR_M * thv[None, :, None] + (kz * z)[:, None, None]
    phi = w(rv)[None, None, :] * np.cos(phase)                       # [Nz][nth][nr+1], unit amplitude
    dth = (np.roll(phi, -1, axis=1) - np.roll(phi, 1, axis=1)) / (2.0 * hth)
    dr = np.empty_like(phi)
    dr[:, :, 1:-1] = (phi[:, :, 2:] - phi[:, :, :-2]) / (2.0 * hr)
    dr[:, :, 0] = (phi[:, :, 1] - phi[:, :, 0]) / hr
    dr[:, :, -1] = (phi[:, :, -1] - phi[:, :, -2]) / hr
    a_p = -dth / rv[None, None, :]
    a_p[:, :, 0] = 0.0
    a_p[:, :, -1] = 0.0
    b_p = dr / rv[None, None, :]
    phi0 = cfl / max(np.abs(a_p).max() * dt / hr, np.abs(b_p).max() * dt / hth)
    a = np.empty((phi.shape[0], nth + 1, nr + 1))
    b = np.empty_like(a)
    for dst, src in ((a, a_p), (b, b_p)):
        dst[:, :nth, :] = phi0 * src
        dst[:, nth, :] = dst[:, 0, :]
    # node values
    r = spec.node_coords(0)
    th = spec.node_coords(1)
    ph = POLAR_M * th[None, :, None] + (kz * z)[:, None, None]
    Ez = phi0 * kz * w(r)[None, None, :] * np.sin(ph)
    xi_r = spec.unit_nodes(0)
    xi_t = spec.unit_nodes(1)
    d0 = phi0 * dth                                                  # [Nz][nth][nr+1] at the vertices
    d1 = np.roll(d0, -1, axis=1)                                     # vertex j+1
    dth_nodes = np.empty((phi.shape[0], nth, len(xi_t), nr, len(xi_r)))
    for q, eta in enumerate(xi_t):
        for p, xi in enumerate(xi_r):
            dth_nodes[:, :, q, :, p] = ((1 - xi) * (1 - eta) * d0[:, :, :-1] + xi * (1 - eta) * d0[:, :, 1:]
                                        + (1 - xi) * eta * d1[:, :, :-1] + xi * eta * d1[:, :, 1:])
    dth_nodes = dth_nodes.reshape(phi.shape[0], nth * len(xi_t), nr * len(xi_r))
    return {"a": a, "b": b, "Ez": np.ascontiguousarray(Ez), "dz_phi": np.ascontiguousarray(-Ez),
            "dth_phi": np.ascontiguousarray(dth_nodes), "phi0": phi0}

"""Pins of the polar delta-g pieces: the theta-only periodic look-up of the tracing, the source
term and mass conservation of the whole step."""
import math

import numpy as np

import oracle
from oracle import polar
from paper_2212_03036_b200 import inputs


def _spec(nx=6, ny=5):
    return inputs.GridSpec(n=(nx, ny, 1, 1), order=(2, 2, 1, 1), lo=(1.0, 0.0, 0.0, 0.0), hi=(4.0, 2 * math.pi, 1.0, 1.0))


def test_theta_only_periodic_lookup_ties_to_the_two_pinned_modes_and_a_closed_form():
    spec = _spec()
    nx, ny = 6, 5
    xv, yv = spec.vertex_coords(0), spec.vertex_coords(1)
    rng = np.random.default_rng(5)
    a = 0.2 * rng.standard_normal((ny + 1, nx + 1))
    b = 0.3 * rng.standard_normal((ny + 1, nx + 1))
    a[-1], b[-1] = a[0], b[0]            # periodic in theta
    a[:, 0] = a[:, -1] = 0.0             # no radial velocity at the radial ends
    tau = 1.1
    # half-step point inside the box along x: same as the fully periodic look-up, bit for bit
    for (i, j, xi, eta) in ((2, 0, 0.3, 0.1), (3, 4, 0.7, 0.95), (1, 4, 0.5, 1.0)):
        assert np.array_equal(oracle.trace(spec, a, b, i, j, xi, eta, tau, 2, 2), oracle.trace(spec, a, b, i, j, xi, eta, tau, 2, 1))
    # half-step point inside the box along theta: same as the clamped look-up
    for (i, j, xi, eta) in ((0, 2, 0.0, 0.5), (5, 2, 1.0, 0.4), (5, 1, 0.9, 0.5)):
        assert np.array_equal(oracle.trace(spec, a, b, i, j, xi, eta, tau, 2, 2), oracle.trace(spec, a, b, i, j, xi, eta, tau, 2, 0))
    # closed form at r_max: a = 0, b linear in r only -> the point slides along theta with b(r_max); a wrapped look-up
    # would take b(r_min) for the half step
    b2 = np.tile(0.1 + 0.25 * xv[None, :], (ny + 1, 1))
    a2 = np.zeros_like(b2)
    foot = oracle.trace(spec, a2, b2, nx - 1, 2, 1.0, 0.25, tau, 2, 2)
    assert abs(foot[0] - 1.0) < 1e-15 and abs(foot[1] - (0.25 - tau * (0.1 + 0.25 * 4.0) / spec.h[1])) < 1e-14
    wrong = oracle.trace(spec, a2, b2, nx - 1, 2, 1.0, 0.25, tau, 2, 1)
    assert abs(wrong[1] - foot[1]) > 0.1


def test_source_step_closed_form_and_mass():
    spec = inputs.polar_grid(6, 8, 3, 8, 2)
    geq, dv, dr = inputs.polar_equilibrium(spec)
    fl = inputs.polar_fields(spec, 4.0)
    f = inputs.polar_initial_dg(spec, eps=0.1)
    out = polar.source_step(f, fl["dz_phi"], fl["dth_phi"], dv, dr, 0.7)
    z, v, y, x = 2, 5, 7, 3
    want = f[z, v, y, x] + 0.7 * (fl["dz_phi"][z, y, x] * dv[v, x] + fl["dth_phi"][z, y, x] * dr[v, x])
    assert abs(out[z, v, y, x] - want) < 1e-18 + 1e-15 * abs(want)
    # analytic derivatives of the Maxwellian (library-free check of the generator): d_v g_eq = -(v/T) g_eq
    r = spec.node_coords(0)
    vv = spec.node_coords(3)
    _, _, T, _ = inputs.polar_profiles(r)
    assert np.allclose(dv, -(vv[:, None] / T[None, :]) * geq, rtol=1e-14)
    h = 1e-5  # d_r(g_eq/r) against a centred difference of f_eq = g_eq / r in r
    n0p, _, Tp, _ = inputs.polar_profiles(r + h)
    n0m, _, Tm, _ = inputs.polar_profiles(r - h)
    fe = lambda n0, T: n0[None, :] / np.sqrt(2 * np.pi * T[None, :]) * np.exp(-vv[:, None] ** 2 / (2 * T[None, :]))
    assert np.allclose(dr, (fe(n0p, Tp) - fe(n0m, Tm)) / (2 * h), rtol=1e-6, atol=1e-12)
    # mass: the v sum of d_v g_eq vanishes by symmetry, the theta Gauss sum of the interpolated centred difference
    # telescopes (section 3.5: "if the derivative is discretized in such a way as to preserve this property")
    m0, m1 = oracle.mass(spec, f), oracle.mass(spec, np.ascontiguousarray(out))
    scale = oracle.mass(spec, np.abs(out - f))
    assert scale > 0 and abs(m1 - m0) < 1e-13 * scale


def test_polar_step_conserves_mass_and_nothing_crosses_the_radial_ends():
    spec = inputs.polar_grid(8, 12, 2, 4, 2)
    geq, dv, dr = inputs.polar_equilibrium(spec)
    dt = 4.0
    fl = inputs.polar_fields(spec, dt, 0.8)
    assert np.all(fl["a"][:, :, 0] == 0.0) and np.all(fl["a"][:, :, -1] == 0.0)
    assert np.array_equal(fl["a"][:, -1], fl["a"][:, 0]) and np.array_equal(fl["b"][:, -1], fl["b"][:, 0])
    # data that hugs both radial ends: a periodic wrap in r would carry mass from one end to the other
    r = spec.node_coords(0)
    f = np.zeros(spec.shape)
    f[:, :, :, :2] = 1.0
    f[:, :, :, -2:] = 2.0
    f *= (1.0 + 0.3 * np.cos(spec.node_coords(1)))[None, None, :, None]
    g = f.copy()
    for _ in range(3):
        g = polar.strang_step_sources(spec, np.ascontiguousarray(g), fl, 0.0 * dv, 0.0 * dr, dt)
    m0, m1 = oracle.mass(spec, f), oracle.mass(spec, np.ascontiguousarray(g))
    assert abs(m1 - m0) < 1e-13 * m0
    # the inner and the outer half keep their own mass (the two ends do not talk to each other)
    half = spec.N[0] // 2
    inner0, inner1 = f.copy(), g.copy()
    inner0[:, :, :, half:] = 0.0
    inner1[:, :, :, half:] = 0.0
    assert abs(oracle.mass(spec, inner1) - oracle.mass(spec, inner0)) < 1e-12 * m0
    # with the equilibrium switched on the source adds no mass either
    g2 = polar.strang_step_sources(spec, inputs.polar_initial_dg(spec, 0.1), fl, dv, dr, dt)
    md = oracle.mass(spec, np.ascontiguousarray(g2)) - oracle.mass(spec, inputs.polar_initial_dg(spec, 0.1))
    assert abs(md) < 1e-13 * oracle.mass(spec, np.abs(g2))


def _polar_manufactured(nr, nth=16, nz=2):
    spec = inputs.GridSpec(n=(nr, nth, nz, 2), order=(2, 2, 2, 2), lo=(0.5, 0.0, 0.0, -1.0), hi=(2.5, 2 * math.pi, 3.0, 1.0))
    rv = spec.vertex_coords(0)
    th = spec.vertex_coords(1)[:-1]
    zeq = (np.arange(spec.N[2]) + 0.5) * spec.h[2] / 2
    R, TH, Z = rv[None, None, :], th[None, :, None], zeq[:, None, None]
    q = math.pi / (2 * 2.0)                      # u(r) = cos(q (r - r_min)): u'(r_min) = 0, u(r_max) = 0
    u, ur, urr = np.cos(q * (R - 0.5)), -q * np.sin(q * (R - 0.5)), -q * q * np.cos(q * (R - 0.5))
    kz = 2 * math.pi / 3.0
    ang = np.cos(3 * TH)
    g = 1.0 + 0.5 * np.cos(kz * Z)               # z profile with mean 1: <phi> = u ang
    dln = 0.3 * np.sin(R)                        # n0'/n0
    Te = 1.0 + 0.2 * R
    rhs = (-(urr + (1.0 / R + dln) * ur) * ang + 9.0 * u * ang / R ** 2) * g + u * ang * (g - 1.0) / Te
    return spec, rhs, dln[0, 0], Te[0, 0], u * ang * g


def test_polar_quasi_neutrality_manufactured_solution_second_order():
    # eq. (2) with Neumann at r_min and Dirichlet at r_max: a dropped 1/r or n0'/n0 term, a wrong
    # theta symbol or a wrong <phi> fails the convergence
    errs = []
    for nr in (16, 32):
        spec, rhs, dln, Te, exact = _polar_manufactured(nr)
        phi = polar.polar_solve_phi(spec, rhs, dln, Te)
        errs.append(np.abs(phi - exact).max())
        assert np.abs(phi[:, :, -1]).max() == 0.0
    assert errs[0] < 5e-3 and 3.5 < errs[0] / errs[1] < 4.5, errs


def test_polar_solver_single_mode_against_a_dense_solve():
    # one (kz, m) mode: the solution stays in that mode and equals the dense solve of the difference equations written
    # out here with numpy.linalg (independent of the banded routine and of the FFT bookkeeping)
    spec = inputs.GridSpec(n=(12, 8, 3, 2), order=(2, 2, 2, 2), lo=(0.3, 0.0, 0.0, -1.0), hi=(2.1, 2 * math.pi, 5.0, 1.0))
    rv = spec.vertex_coords(0)
    th = spec.vertex_coords(1)[:-1]
    zeq = (np.arange(spec.N[2]) + 0.5) * spec.h[2] / 2
    prof = np.sin(1.7 * rv) + 0.3
    m, kzi = 2, 1
    rhs = prof[None, None, :] * np.cos(m * th[None, :, None] + 2 * math.pi * kzi * zeq[:, None, None] / 5.0)
    dln, Te = 0.2 * rv, 0.7 + 0.1 * rv
    phi = polar.polar_solve_phi(spec, rhs, dln, Te)
    nr, h = 12, spec.h[0]
    M = np.zeros((nr, nr))
    for i in range(nr):
        adv = (1.0 / rv[i] + dln[i]) / (2 * h)
        M[i, i] = 2 / h ** 2 + m * m / rv[i] ** 2 + 1.0 / Te[i]
        if i + 1 < nr:
            M[i, i + 1] = -1 / h ** 2 - adv
        if i > 0:
            M[i, i - 1] = -1 / h ** 2 + adv
        else:
            M[0, 1] += -1 / h ** 2 + adv
    amp = np.concatenate([np.linalg.solve(M, prof[:nr]), [0.0]])
    want = amp[None, None, :] * np.cos(m * th[None, :, None] + 2 * math.pi * kzi * zeq[:, None, None] / 5.0)
    assert np.abs(phi - want).max() < 1e-12 * np.abs(want).max()


def test_polar_resampling_and_derived_fields():
    spec = inputs.polar_grid(6, 8, 3, 4, 2)
    r, th, z = spec.node_coords(0), spec.node_coords(1), spec.node_coords(2)
    rho = (1.0 + 0.01 * z)[:, None, None] * (2.0 + 0.1 * r)[None, None, :] * np.ones_like(th)[None, :, None]
    out = polar.polar_resample(spec, rho)
    rv = spec.vertex_coords(0)
    zeq = (np.arange(spec.N[2]) + 0.5) * spec.h[2] / 2
    want = (1.0 + 0.01 * zeq)[:, None, None] * (2.0 + 0.1 * rv)[None, None, :] * np.ones(8)[None, :, None]
    assert np.abs(out - want).max() < 1e-12      # linear in r: exact at every vertex, the radial ends included
    # derived fields of one Fourier mode: centred differences multiply by sin(k h)/h; radial ends of a are zero
    thv = spec.vertex_coords(1)[:-1]
    phi = (np.sin(rv)[None, None, :] * np.cos(3 * thv[None, :, None] + 2 * math.pi * zeq[:, None, None] / spec.hi[2]))
    a, b, e, dth = polar.polar_derive(spec, phi)
    hth, hz = spec.h[1], spec.h[2] / 2
    ph = 3 * thv[None, :, None] + 2 * math.pi * zeq[:, None, None] / spec.hi[2]
    assert np.abs(dth - (-np.sin(3 * hth) / hth * np.sin(rv)[None, None, :] * np.sin(ph))).max() < 1e-12
    assert np.abs(a[:, :, 1:-1] - (-dth / rv[None, None, :])[:, :, 1:-1]).max() < 1e-15
    assert np.all(a[:, :, 0] == 0.0) and np.all(a[:, :, -1] == 0.0) and np.all(b[:, :, 0] == 0.0)
    kz = 2 * math.pi / spec.hi[2]
    assert np.abs(e - (np.sin(kz * hz) / hz * np.sin(rv)[None, None, :] * np.sin(ph))).max() < 1e-12
    h = spec.h[0]
    assert np.abs(b[:, :, 3] - (phi[:, :, 4] - phi[:, :, 2]) / (2 * h) / rv[3]).max() < 1e-15


def test_polar_algorithms_differ_by_a_local_second_order_term():
    # as in the Cartesian case: one step of Algorithm 1 and one of Algorithm 2 from the same state differ
    # by O(dt^2) -- the field of Algorithm 1's second half is a first-order approximation of phi^{n+1/2}
    spec = inputs.polar_grid(12, 16, 4, 12, 2)
    rv = spec.vertex_coords(0)
    n0, dln_n0, T, _ = inputs.polar_profiles(rv)
    _, dv, dr = inputs.polar_equilibrium(spec)
    dg0 = inputs.polar_initial_dg(spec, eps=0.05)
    m0 = oracle.mass(spec, dg0)
    d = []
    for dt in (4.0, 2.0, 1.0):
        g1, _ = polar.polar_algorithm1_step(spec, dg0.copy(), n0, dln_n0, T, dv, dr, dt)
        g2, _ = polar.polar_algorithm2_step(spec, dg0.copy(), n0, dln_n0, T, dv, dr, dt)
        d.append(np.abs(g1 - g2).max())
        scale = oracle.mass(spec, np.abs(g2))
        assert abs(oracle.mass(spec, np.ascontiguousarray(g2)) - m0) < 1e-13 * scale
    assert 1.8 < math.log2(d[0] / d[1]) < 2.2 and 1.8 < math.log2(d[1] / d[2]) < 2.2, d

"""Pins of the field-step oracle (oracle/field.py; eq. (2), :281-283): closed forms and
invariants chosen so that a dropped term, a wrong sign or index, or a wrong scale fails one of them."""
import math

import numpy as np
import pytest

from oracle import field
from paper_2212_03036_b200 import inputs


def _spec(nx, ny, nz, o=2, nv=2):
    return inputs.GridSpec(n=(nx, ny, nz, nv), order=(o, o, o, o), lo=(-1.0, 0.5, 0.0, -2.0), hi=(2.0, 2.5, 7.0, 2.0))


@pytest.mark.parametrize("o", [1, 2, 3])
def test_resampling_is_exact_for_polynomials_of_degree_below_o(o):
    # a global polynomial of per-variable degree < o is its own nodal interpolant in every cell: the resampled values
    # are the function's values at the vertices (interior) and at the equidistant z points; at the periodic seam a
    # vertex sees the mean of the function's values at both ends of the box ("the average is taken")
    spec = _spec(5, 4, 3, o)
    c1, c2 = float(o > 1), float(o > 2)
    px = lambda x: 1.0 + c1 * 0.3 * x + c2 * 0.05 * x * x
    py = lambda y: 2.0 - c1 * 0.1 * y + c2 * 0.02 * y * y
    pz = lambda z: 1.0 + c1 * 0.01 * z - c2 * 0.003 * z * z
    x, y, z = spec.node_coords(0), spec.node_coords(1), spec.node_coords(2)
    rho = pz(z)[:, None, None] * py(y)[None, :, None] * px(x)[None, None, :]
    out = field.resample_rho(spec, rho)
    xv, yv = spec.vertex_coords(0), spec.vertex_coords(1)
    zeq = spec.lo[2] + (np.arange(spec.N[2]) + 0.5) * spec.h[2] / o
    fx = px(xv[:-1]).copy()
    fx[0] = 0.5 * (px(xv[0]) + px(xv[-1]))
    fy = py(yv[:-1]).copy()
    fy[0] = 0.5 * (py(yv[0]) + py(yv[-1]))
    want = pz(zeq)[:, None, None] * fy[None, :, None] * fx[None, None, :]
    assert np.abs(out - want).max() < 1e-13


def _fourier_solution(spec, rhs, T0):
    """Closed form for constant n0 and Te = T0: the discrete operator is diagonal in the Fourier basis, symbol
    (4/hx^2) sin^2(pi kx/nx) + (4/hy^2) sin^2(pi ky/ny), plus 1/T0 on the modes with kz != 0 (<phi> removes kz = 0)."""
    Nz, ny, nx = rhs.shape
    hx, hy = spec.h[0], spec.h[1]
    R = np.fft.fftn(rhs)
    kx = np.arange(nx)[None, None, :]
    ky = np.arange(ny)[None, :, None]
    kz = np.arange(Nz)[:, None, None]
    lam = 4.0 / hx ** 2 * np.sin(math.pi * kx / nx) ** 2 + 4.0 / hy ** 2 * np.sin(math.pi * ky / ny) ** 2
    sym = lam + (kz != 0) / T0
    sym[0, 0, 0] = 1.0
    P = R / sym
    P[0, 0, 0] = 0.0  # compatibility projection and zero-mean gauge
    return np.real(np.fft.ifftn(P))


def test_constant_coefficients_reduce_to_the_fourier_symbol():
    spec = _spec(8, 6, 5)
    rng = np.random.default_rng(7)
    rhs = rng.standard_normal((spec.N[2], 6, 8))
    n0 = np.full((6, 8), 1.7)
    Te = np.full((6, 8), 0.8)
    phi, pbar = field.solve_phi(spec, rhs, n0, Te)
    want = _fourier_solution(spec, rhs, 0.8)
    assert np.abs(phi - want).max() < 1e-11 * np.abs(want).max()
    assert np.abs(pbar - want.mean(axis=0)).max() < 1e-11 * np.abs(want).max()


def test_z_independent_source_gives_z_independent_potential_without_the_Te_term():
    # phi = <phi>: the adiabatic term vanishes and A phi = rhs - c alone decides (R21, R22)
    spec = _spec(6, 6, 2)
    rng = np.random.default_rng(3)
    n0 = 1.0 + 0.3 * rng.random((6, 6))
    Te = 0.5 + rng.random((6, 6))
    r2 = rng.standard_normal((6, 6))
    rhs = np.repeat(r2[None], spec.N[2], axis=0)
    phi, pbar = field.solve_phi(spec, rhs, n0, Te)
    assert np.abs(phi - pbar[None]).max() < 1e-12
    assert abs(pbar.sum()) < 1e-12
    A = field.assemble_A(spec, n0)
    c = (n0 * r2).sum() / n0.sum()
    assert np.abs(A @ pbar.reshape(-1) - (r2.reshape(-1) - c)).max() < 1e-11
    # the same potential whatever Te is
    phi2, _ = field.solve_phi(spec, rhs, n0, 3.0 * Te)
    assert np.abs(phi2 - phi).max() < 1e-12


def _manufactured(n, nz=2):
    spec = inputs.GridSpec(n=(n, n, nz, 2), order=(2, 2, 2, 2), lo=(0.0, 0.0, 0.0, -1.0), hi=(2.0, 3.0, 5.0, 1.0))
    Lx, Ly, Lz = 2.0, 3.0, 5.0
    kx, ky, kz = 2 * math.pi / Lx, 2 * math.pi / Ly, 2 * math.pi / Lz
    xv, yv = spec.vertex_coords(0)[:-1], spec.vertex_coords(1)[:-1]
    zeq = (np.arange(spec.N[2]) + 0.5) * spec.h[2] / 2
    X, Y, Z = xv[None, None, :], yv[None, :, None], zeq[:, None, None]
    g = 1.0 + 0.5 * np.cos(kz * Z)                      # z profile, mean 1
    u = np.sin(kx * X) * np.cos(ky * Y)                 # phi = u g, zero mean over the plane
    ux, uy = kx * np.cos(kx * X) * np.cos(ky * Y), -ky * np.sin(kx * X) * np.sin(ky * Y)
    lap = -(kx ** 2 + ky ** 2) * u
    n0 = 1.0 + 0.3 * np.cos(kx * X) * np.sin(ky * Y)
    n0x, n0y = -0.3 * kx * np.sin(kx * X) * np.sin(ky * Y), 0.3 * ky * np.cos(kx * X) * np.cos(ky * Y)
    Te = 1.0 + 0.2 * np.sin(ky * Y) + 0.0 * X
    # -(1/n0) div(n0 grad phi) + (phi - <phi>)/Te  with <phi> = u (the z mean of g is 1)
    rhs = -(n0x * ux + n0y * uy + n0 * lap) / n0 * g + u * (g - 1.0) / Te
    return spec, rhs, n0[0], Te[0], u * g


def test_manufactured_solution_converges_at_second_order():
    errs = []
    for n in (16, 32):
        spec, rhs, n0, Te, exact = _manufactured(n)
        phi, _ = field.solve_phi(spec, rhs, n0, Te)
        # gauge: the exact <phi> has zero mean over the plane, and so has the discrete one
        errs.append(np.abs(phi - exact).max())
    assert errs[0] < 2e-2
    assert 3.5 < errs[0] / errs[1] < 4.5, errs


def test_derived_fields_have_the_drift_signs_and_the_difference_symbols():
    # one Fourier mode: centred differences multiply by i sin(k h)/h exactly
    spec = _spec(12, 10, 4)
    xv, yv = spec.vertex_coords(0)[:-1], spec.vertex_coords(1)[:-1]
    zeq = (np.arange(spec.N[2]) + 0.5) * spec.h[2] / 2
    kx, ky, kz = 2 * math.pi / 3.0, 2 * math.pi * 2 / 2.0, 2 * math.pi / 7.0
    ph = kx * xv[None, None, :] + ky * yv[None, :, None] + kz * zeq[:, None, None]
    a, b, e = field.derive_fields(spec, np.sin(ph), B=2.0)
    hx, hy, hz = spec.h[0], spec.h[1], spec.h[2] / 2
    assert np.abs(a - (-np.sin(ky * hy) / hy * np.cos(ph) / 2.0)).max() < 1e-12   # a = -d_y phi / B
    assert np.abs(b - (np.sin(kx * hx) / hx * np.cos(ph) / 2.0)).max() < 1e-12    # b = +d_x phi / B
    assert np.abs(e - (-np.sin(kz * hz) / hz * np.cos(ph))).max() < 1e-12         # E = -d_z phi


def test_interpolation_to_the_nodes_reproduces_linear_functions():
    spec = _spec(5, 4, 3, 3)
    xv, yv = spec.vertex_coords(0)[:-1], spec.vertex_coords(1)[:-1]
    zeq = spec.lo[2] + (np.arange(spec.N[2]) + 0.5) * spec.h[2] / 3
    F = 0.3 + 0.7 * xv[None, None, :] - 0.2 * yv[None, :, None] + 0.05 * zeq[:, None, None]
    x, y, z = spec.node_coords(0), spec.node_coords(1), spec.node_coords(2)
    G = field.xy_to_nodes(spec, F)
    want = 0.3 + 0.7 * x[None, None, :] - 0.2 * y[None, :, None] + 0.05 * zeq[:, None, None]
    inner = (slice(None), slice(0, 3 * 3), slice(0, 4 * 3))  # cells not touching the periodic seam
    assert np.abs(G[inner] - want[inner]).max() < 1e-13
    H = field.z_to_nodes(spec, G)
    want = 0.3 + 0.7 * x[None, None, :] - 0.2 * y[None, :, None] + 0.05 * z[:, None, None]
    zin = (z > zeq[0]) & (z < zeq[-1])  # between two field points of the same period
    assert np.abs(H[zin][:, :9, :12] - want[zin][:, :9, :12]).max() < 1e-13
    W = field.with_wrap(F)
    assert np.array_equal(W[:, -1, :], W[:, 0, :]) and np.array_equal(W[:, :, -1], W[:, :, 0])
    assert np.array_equal(W[:, :-1, :-1], F)


def test_diagnostics_closed_forms():
    spec = inputs.GridSpec(n=(8, 8, 3, 4), order=(2, 2, 2, 2), lo=(-2.0, -2.0, 0.0, -3.0), hi=(2.0, 2.0, 6.0, 3.0))
    v = spec.node_coords(3)
    x = spec.node_coords(0)
    f = np.empty(spec.shape)
    f[...] = (1.0 + 0.5 * v)[None, :, None, None] * (2.0 + x)[None, None, None, :]
    phi = np.full((spec.N[2], 8, 8), 0.25)
    d = field.diagnostics(spec, f, phi, np.full((spec.N[2], 16, 16), 0.25), 1.3)
    vol_yz = 4.0 * 6.0
    ix = 2.0 * 4.0            # int (2 + x) dx over [-2, 2]
    ix2 = 4.0 * 4.0 + 16 / 3  # int (2 + x)^2
    assert abs(d["mass"] - vol_yz * ix * 6.0) < 1e-11
    assert abs(d["kinetic"] - vol_yz * ix * 0.5 * 18.0) < 1e-11           # int v^2/2 (1 + v/2) dv = 9
    assert abs(d["l2"] - math.sqrt(vol_yz * ix2 * (6.0 + 0.25 * 18.0))) < 1e-11
    assert abs(d["potential"] - 0.25 * d["mass"]) < 1e-11
    assert abs(d["electric"] - 0.25 * math.sqrt(2 * math.pi * 6.0)) < 1e-12


def _small_itg():
    spec = inputs.itg_grid(12, 12, 4, 12, 2)
    n0, Te = inputs.itg_vertex_profiles(spec)
    return spec, n0, Te, inputs.itg_initial_f(spec, eps=0.3)


def test_algorithms_1_and_2_differ_by_a_local_second_order_term_and_conserve_mass():
    # Algorithm 1 "fails to be second order because the electric field that is used to trace the
    # characteristics is not a sufficiently accurate approximation at half the time step" -- its field phi* is an O(dt)
    # approximation of phi^{n+1/2}, so one step of Algorithm 1 and one of Algorithm 2 differ by O(dt^2) (the spatial
    # projection errors, identical substeps, cancel): halving dt divides the difference by 4
    import oracle
    spec, n0, Te, f0 = _small_itg()
    m0 = oracle.mass(spec, f0)
    d = []
    for dt in (4.0, 2.0, 1.0):
        f1, _ = field.algorithm1_step(spec, f0.copy(), n0, Te, dt)
        f2, _ = field.algorithm2_step(spec, f0.copy(), n0, Te, dt)
        d.append(np.abs(f1 - f2).max())
        assert abs(oracle.mass(spec, f1) - m0) < 1e-13 * m0 and abs(oracle.mass(spec, f2) - m0) < 1e-13 * m0
    assert 1.85 < math.log2(d[0] / d[1]) < 2.15 and 1.85 < math.log2(d[1] / d[2]) < 2.15, d


def test_algorithm_steps_are_the_papers_sequences():
    # the order of Algorithm 1 (steps 1, 3-8) and of Algorithm 2 (1, 3-6, 8-12) written out with the pinned substeps
    import oracle
    spec, n0, Te, f0 = _small_itg()
    dt = 3.0
    fs = field.field_step(spec, oracle.charge_density(spec, f0), n0, Te)
    g = oracle.advect_v(spec, oracle.advect_z(spec, f0, dt / 2), fs["Ez"], dt / 2)
    fs1 = field.field_step(spec, oracle.charge_density(spec, g), n0, Te)
    w1 = oracle.advect_z(spec, oracle.advect_v(spec, oracle.advect_xy(spec, g, fs1["a"], fs1["b"], dt, 2, 1), fs1["Ez"], dt / 2), dt / 2)
    got1, _ = field.algorithm1_step(spec, f0.copy(), n0, Te, dt)
    assert np.array_equal(got1, w1)
    half = oracle.advect_xy(spec, g, fs["a"], fs["b"], dt / 2, 1, 1)                # predictor: eq. (14), dt/2, phi^n
    fs2 = field.field_step(spec, oracle.charge_density(spec, half), n0, Te)
    h = oracle.advect_v(spec, oracle.advect_z(spec, f0, dt / 2), fs2["Ez"], dt / 2)  # corrector restarts from f^n
    w2 = oracle.advect_z(spec, oracle.advect_v(spec, oracle.advect_xy(spec, h, fs2["a"], fs2["b"], dt, 2, 1), fs2["Ez"], dt / 2), dt / 2)
    got2, _ = field.algorithm2_step(spec, f0.copy(), n0, Te, dt)
    assert np.array_equal(got2, w2)


def test_algorithm2_is_second_order_in_time_where_algorithm1_is_not():
    # "We propose the second order scheme in algorithm 2".  A smooth low-mode state with constant
    # profiles (so that the spatial error is small against the temporal one at these step sizes), T = 1.6 with dt = 0.8,
    # 0.4, 0.2: the successive differences shrink by ~2^2 for Algorithm 2 and by ~2^1.3 for Algorithm 1.  (Finer steps meet
    # the h^{k+1}/dt term of semi-Lagrangian schemes: measured orders 1.27-1.50 from dt = 0.2 to 0.1 on 8^2-20^2 cells.)
    spec = inputs.GridSpec(n=(8, 8, 10, 24), order=(3, 3, 3, 3), lo=(0, 0, 0, -4.0), hi=(2 * math.pi, 2 * math.pi, 2 * math.pi, 4.0))
    x, y, z, v = (spec.node_coords(d) for d in range(4))
    f0 = (np.exp(-0.5 * v * v) / math.sqrt(2 * math.pi))[None, :, None, None] * (
        1 + 0.3 * np.cos(x)[None, None, None, :] * np.cos(y[None, None, :, None] + z[:, None, None, None]))
    f0 = np.ascontiguousarray(f0)
    n0 = np.ones((8, 8))
    Te = np.ones((8, 8))

    def run(alg, dt):
        f = f0.copy()
        for _ in range(int(round(1.6 / dt))):
            f, _ = alg(spec, f, n0, Te, dt)
        return f

    orders = {}
    for name, alg in (("alg1", field.algorithm1_step), ("alg2", field.algorithm2_step)):
        sols = [run(alg, dt) for dt in (0.8, 0.4, 0.2)]
        d = [np.abs(sols[i] - sols[i + 1]).max() for i in range(2)]
        orders[name] = math.log2(d[0] / d[1])
    assert orders["alg2"] > 1.75 and orders["alg1"] < 1.5, orders

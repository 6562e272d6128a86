"""Pins for the 1d part of the CPU oracle (oracle/sldg_oracle.c): Gauss-Legendre tables, the overlap
matrices A(alpha), B(alpha) of eq. (11), the periodic line shift, the 4d z- and v-sweeps
(eq. 4-5), charge density and mass.

Each pin is something the paper or the mathematics fixes, computed WITHOUT the oracle: golden values
from an independent CAS derivation, invariants, closed forms, numpy library routines, and a brute-force
L2 projection of the shifted piecewise polynomial.  No GPU needed.
"""
import os

import numpy as np
import pytest

import oracle
from paper_2212_03036_b200.inputs import GridSpec

ORDERS = [1, 2, 3, 4]


def _lag(nodes, j, x):
    v = np.ones_like(x, dtype=np.float64)
    for i, xi in enumerate(nodes):
        if i != j:
            v = v * (x - xi) / (nodes[j] - xi)
    return v


def _np_gl(o):
    t, w = np.polynomial.legendre.leggauss(o)
    return 0.5 * (t + 1.0), 0.5 * w


# ---------------------------------------------------------------------------------------------- GL
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 8, 12])
def test_gl_matches_numpy_leggauss(n):
    x, w = oracle.gl(n)
    xr, wr = _np_gl(n)
    assert np.allclose(x, xr, rtol=0, atol=2e-16 * 4)
    assert np.allclose(w, wr, rtol=0, atol=1e-15)
    # exact for monomials up to degree 2n-1 on (0,1)
    for d in range(2 * n):
        assert abs(np.dot(w, x ** d) - 1.0 / (d + 1)) < 1e-15


# ------------------------------------------------------------------------------- overlap matrices
def _golden_shift(golden_dir):
    rows = {}
    with open(os.path.join(golden_dir, "shift_matrices.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            o, alpha, name, r, c, val = line.split()
            rows.setdefault((int(o), float(alpha)), []).append((name, int(r), int(c), float(val)))
    return rows


def test_shift_matrices_golden(golden_dir):
    """SURVEY.md 8(c)-1 printed values (independent CAS derivation of eq. 10)."""
    gold = _golden_shift(golden_dir)
    assert len(gold) == 3
    for (o, alpha), entries in gold.items():
        A, B = oracle.shift_matrices(o, alpha)
        assert len(entries) == 2 * o * o
        for name, r, c, val in entries:
            got = (A if name == "A" else B)[r, c]
            assert abs(got - val) < 5e-16, (o, alpha, name, r, c, got, val)


def test_shift_matrices_closed_form_o2():
    """Closed form for o=2 from SURVEY.md 8(c)-1 (polynomials in alpha), at many alpha."""
    s3 = np.sqrt(3.0)
    for al in np.linspace(0.0, 1.0, 41)[:-1]:
        A, B = oracle.shift_matrices(2, al)
        Ar = np.array([[al ** 3 - 2 * al + 1, al * (-al ** 2 - s3 * al + 1 + s3)],
                       [al * (-al ** 2 + s3 * al - s3 + 1), al ** 3 - 2 * al + 1]])
        Br = np.array([[al * (-al ** 2 + 3 * al - 1), al * (al ** 2 - 3 * al + s3 * al - s3 + 2)],
                       [al * (al ** 2 - 3 * al - s3 * al + s3 + 2), al * (-al ** 2 + 3 * al - 1)]])
        assert np.abs(A - Ar).max() < 4e-16
        assert np.abs(B - Br).max() < 4e-16


@pytest.mark.parametrize("o", ORDERS)
def test_shift_matrices_invariants(o):
    x, w = _np_gl(o)
    A0, B0 = oracle.shift_matrices(o, 0.0)
    # integer Courant numbers are exact copies: A(0) = I, B(0) = 0 bit for bit
    assert np.array_equal(A0, np.eye(o)) and np.array_equal(B0, np.zeros((o, o)))
    J = np.eye(o)[::-1]
    for al in [1e-9, 0.1, 0.25, 1.0 / 3.0, 0.5, 0.77, 1.0 - 1e-9]:
        A, B = oracle.shift_matrices(o, al)
        assert np.abs((A + B) @ np.ones(o) - 1.0).max() < 1e-14        # constants preserved
        assert np.abs(w @ (A + B) - w).max() < 1e-15                   # mass
        A1, B1 = oracle.shift_matrices(o, 1.0 - al)
        assert np.abs(B - J @ A1 @ J).max() < 1e-14                    # mirror symmetry
    # continuity across the floor branch: A(alpha) -> 0, B(alpha) -> I as alpha -> 1
    A, B = oracle.shift_matrices(o, 1.0 - 1e-12)
    assert np.abs(A).max() < 1e-10 and np.abs(B - np.eye(o)).max() < 1e-10


def _brute_shift(u, o, delta, nq=12):
    """Definition (eq. 10): u+ = L2-projection of u(. - delta) -- direct quadrature of
    the shifted piecewise polynomial, split at its break point.  Independent of the oracle."""
    n = u.size // o
    xn, wn = _np_gl(o)
    xq, wq = _np_gl(nq)

    def upw(x):
        x = np.mod(x, n)
        c = np.minimum(np.floor(x).astype(int), n - 1)
        loc = x - c
        val = np.zeros_like(x)
        for m in range(o):
            val += u[c * o + m] * _lag(xn, m, loc)
        return val

    out = np.empty_like(u)
    brk = delta - np.floor(delta)  # xi where i + xi - delta crosses a cell boundary
    pieces = [(0.0, brk), (brk, 1.0)]
    for i in range(n):
        for j in range(o):
            acc = 0.0
            for (lo, hi) in pieces:
                if hi - lo <= 0:
                    continue
                xi = lo + (hi - lo) * xq
                # nudge evaluation points strictly inside the piece (they are: GL nodes are interior)
                acc += (hi - lo) * np.dot(wq, _lag(xn, j, xi) * upw(i + xi - delta))
            out[i * o + j] = acc / wn[j]
    return out


@pytest.mark.parametrize("o", ORDERS)
@pytest.mark.parametrize("delta", [0.3, -0.3, 0.999, -1.25, 2.6, -7.45, 13.5, 1e-7])
def test_line_shift_matches_bruteforce_projection(o, delta):
    rng = np.random.default_rng(100 + o)
    n = 7
    u = rng.standard_normal(n * o)
    got = oracle.shift_line(u, o, delta)
    ref = _brute_shift(u, o, delta)
    assert np.abs(got - ref).max() < 2e-13


@pytest.mark.parametrize("o", ORDERS)
@pytest.mark.parametrize("k", [0, 1, -1, 3, -4, 9, -23])
def test_line_shift_integer_courant_is_exact_roll(o, k):
    """u+(x) = u(x - a tau): delta = +k moves data k cells to the right, bit for bit, with wrap."""
    rng = np.random.default_rng(7)
    n = 6
    u = rng.standard_normal(n * o)
    got = oracle.shift_line(u, o, float(k))
    ref = np.roll(u.reshape(n, o), k, axis=0).reshape(-1)
    assert np.array_equal(got, ref)


@pytest.mark.parametrize("o", [2, 3, 4])
def test_line_shift_polynomial_exactness(o):
    """A global polynomial of degree < o is transported exactly (cells whose sources do not wrap)."""
    n = 12
    xn, _ = _np_gl(o)
    x = (np.arange(n)[:, None] + xn[None, :]).reshape(-1)
    coef = np.array([0.7, -1.3, 0.45, 0.21])[:o]
    poly = lambda t: sum(c * t ** d for d, c in enumerate(coef))
    for delta in [0.37, -0.81, 2.25, -3.6]:
        got = oracle.shift_line(poly(x), o, delta).reshape(n, o)
        ref = poly(x - delta).reshape(n, o)
        lo = int(np.ceil(max(delta, 0))) + 1
        hi = n - int(np.ceil(max(-delta, 0))) - 1
        assert np.abs(got[lo:hi] - ref[lo:hi]).max() < 1e-12 * max(1.0, np.abs(ref).max())


@pytest.mark.parametrize("o", ORDERS)
def test_line_shift_mass_and_momentum(o):
    """Mass is conserved; with compact data the first moment moves by delta * mass."""
    n = 16
    xn, wn = _np_gl(o)
    x = (np.arange(n)[:, None] + xn[None, :])
    rng = np.random.default_rng(3)
    u = np.zeros((n, o))
    u[6:9] = rng.standard_normal((3, o))  # compact support away from the periodic seam
    for delta in [0.41, -1.73, 2.5]:
        up = oracle.shift_line(u.reshape(-1), o, delta).reshape(n, o)
        m0, m1 = (u * wn).sum(), (up * wn).sum()
        assert abs(m1 - m0) < 1e-14
        p0, p1 = (u * wn * x).sum(), (up * wn * x).sum()
        if o >= 2:
            assert abs(p1 - (p0 + delta * m0)) < 1e-13
    # random periodic data: mass only
    u = rng.standard_normal((n, o))
    up = oracle.shift_line(u.reshape(-1), o, 5.37).reshape(n, o)
    assert abs((up * wn).sum() - (u * wn).sum()) < 1e-13


# ------------------------------------------------------------------------------------- 4d sweeps
def _small_spec(o=2, n=(3, 2, 5, 4)):
    return GridSpec(n=n, order=(o, o, o, o), lo=(-1.0, -2.0, 0.0, -3.0), hi=(1.0, 2.0, 10.0, 3.0))


@pytest.mark.parametrize("o", [2, 3])
def test_advect_z_lines_and_speeds(o):
    """Every (v,y,x) column is the 1d shift with Courant number v_q tau / h_z, v_q the NODE value
    (reading A2; eq. 4).  The per-line reference is the brute-force projection."""
    spec = _small_spec(o)
    rng = np.random.default_rng(11)
    f = rng.standard_normal(spec.shape)
    tau = 1.9
    got = oracle.advect_z(spec, f, tau)
    v = spec.node_coords(3)
    hz = spec.h[2]
    Nz, Nv, Ny, Nx = spec.shape
    for V in range(Nv):
        for (Y, X) in [(0, 0), (Ny - 1, Nx - 1), (1, 2)]:
            ref = _brute_shift(f[:, V, Y, X].copy(), o, v[V] * tau / hz)
            assert np.abs(got[:, V, Y, X] - ref).max() < 1e-12


@pytest.mark.parametrize("o", [2, 3])
def test_advect_v_lines_and_speeds(o):
    """Every (z,y,x) line is the 1d shift with Courant number Ez tau / h_v, periodic in v
    (readings A3, A4; eq. 5)."""
    spec = _small_spec(o)
    rng = np.random.default_rng(12)
    f = rng.standard_normal(spec.shape)
    Nz, Nv, Ny, Nx = spec.shape
    Ez = rng.uniform(-4.0, 4.0, size=(Nz, Ny, Nx))
    tau = 0.8
    got = oracle.advect_v(spec, f, Ez, tau)
    hv = spec.h[3]
    for (Z, Y, X) in [(0, 0, 0), (Nz - 1, Ny - 1, Nx - 1), (2, 1, 3), (4, 3, 1)]:
        ref = _brute_shift(f[Z, :, Y, X].copy(), o, Ez[Z, Y, X] * tau / hv)
        assert np.abs(got[Z, :, Y, X] - ref).max() < 1e-12


def test_advect_z_integer_courant_rolls_planes():
    """Uniform v grid chosen so that every node speed gives an integer Courant number is impossible
    (nodes are GL points); use order 1 in v so the node is the cell centre."""
    spec = GridSpec(n=(2, 2, 6, 4), order=(2, 2, 2, 1), lo=(0, 0, 0.0, -2.0), hi=(1, 1, 6.0, 2.0))
    rng = np.random.default_rng(5)
    f = rng.standard_normal(spec.shape)
    v = spec.node_coords(3)  # -1.5, -0.5, 0.5, 1.5
    tau = 2.0                # hz = 1 -> Courant numbers -3, -1, 1, 3
    got = oracle.advect_z(spec, f, tau)
    Nz, Nv, Ny, Nx = spec.shape
    for V in range(Nv):
        k = int(round(v[V] * tau))
        ref = np.roll(f[:, V].reshape(6, 2, Ny, Nx), k, axis=0).reshape(Nz, Ny, Nx)
        assert np.array_equal(got[:, V], ref)


def test_charge_density_and_mass_closed_form():
    """GL sums integrate the DG polynomial exactly: separable polynomial data -> closed forms."""
    spec = GridSpec(n=(3, 4, 2, 5), order=(2, 2, 2, 2), lo=(-1.0, 0.0, 0.0, -2.0), hi=(2.0, 1.0, 4.0, 3.0))
    x, y, z, v = (spec.node_coords(d) for d in range(4))
    # degree <= 3 per variable is integrated exactly by the 2-point rule per cell
    f = ((1 + x ** 3)[None, None, None, :] * (2 - y ** 2)[None, None, :, None]
         * (1 + 0.5 * z)[:, None, None, None] * (v ** 2 + v ** 3)[None, :, None, None])
    rho = oracle.charge_density(spec, f)
    iv = (3.0 ** 3 - (-2.0) ** 3) / 3 + (3.0 ** 4 - (-2.0) ** 4) / 4
    ref = iv * (1 + x ** 3)[None, None, :] * (2 - y ** 2)[None, :, None] * (1 + 0.5 * z)[:, None, None]
    assert np.abs(rho - ref).max() < 1e-12 * np.abs(ref).max()
    ix = (2.0 - (-1.0)) + (2.0 ** 4 - 1.0) / 4
    iy = 2.0 - 1.0 / 3
    iz = 4.0 + 0.25 * 16.0
    assert abs(oracle.mass(spec, f) - ix * iy * iz * iv) < 1e-12 * abs(ix * iy * iz * iv)


def test_sweeps_conserve_mass():
    spec = _small_spec(2, n=(3, 3, 6, 6))
    rng = np.random.default_rng(21)
    f = rng.random(spec.shape)
    Nz, Nv, Ny, Nx = spec.shape
    Ez = rng.uniform(-3, 3, size=(Nz, Ny, Nx))
    m0 = oracle.mass(spec, f)
    f1 = oracle.advect_z(spec, f, 3.3)
    f2 = oracle.advect_v(spec, f1, Ez, 0.9)
    assert abs(oracle.mass(spec, f1) - m0) < 1e-14 * abs(m0)
    assert abs(oracle.mass(spec, f2) - m0) < 1e-14 * abs(m0)

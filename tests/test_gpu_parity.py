"""Parity of the CUDA path (libsldg through the C-ABI) against the CPU oracle, element by element on the
same seeded inputs.  Bar (north_star): relative L-infinity error <= 1e-11, mass conserved to <= 1e-13
relative; integer/index work (integer Courant numbers, layout transposes) bit-exact."""
import math

import numpy as np
import pytest

import oracle
from paper_2212_03036_b200 import inputs
from paper_2212_03036_b200.inputs import GridSpec

pytestmark = pytest.mark.gpu

TOL = 1e-11


@pytest.fixture(scope="module")
def torch():
    import torch as t
    if not t.cuda.is_available():
        pytest.skip("needs a CUDA device")
    return t


def _sldg(spec, layout=0):
    from paper_2212_03036_b200.binding import Sldg
    return Sldg(spec, layout=layout)


def _dev(torch, x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def _rel(got, ref):
    return np.abs(got - ref).max() / np.abs(ref).max()


SPECS = {
    "o2_ragged": GridSpec(n=(5, 3, 7, 11), order=(2, 2, 2, 2), lo=(-1, -2, 0, -3.0), hi=(1, 2, 10, 3.5)),
    "o3_ragged": GridSpec(n=(4, 5, 6, 7), order=(3, 3, 3, 3), lo=(-1, -2, 0, -3.0), hi=(1, 2, 10, 3.5)),
    "mixed": GridSpec(n=(6, 4, 5, 40), order=(2, 2, 3, 2), lo=(0, 0, 0, -2.0), hi=(1, 1, 5, 2.0)),
    "o1": GridSpec(n=(6, 4, 9, 70), order=(2, 2, 1, 1), lo=(0, 0, 0, -2.0), hi=(1, 1, 5, 2.0)),
}


@pytest.mark.parametrize("name", list(SPECS))
@pytest.mark.parametrize("layout", [1, 2, 3])
def test_pack_unpack_roundtrip_is_bit_exact(torch, name, layout):
    spec = SPECS[name]
    rng = np.random.default_rng(1)
    f = rng.standard_normal(spec.shape)
    s = _sldg(spec, layout)
    s.import_state(_dev(torch, f))
    out = s.export_state().cpu().numpy()
    s.check()
    assert np.array_equal(out, f)
    host = np.empty_like(f)
    s.import_state_host(f)
    s.export_state_host(host)
    assert np.array_equal(host, f)


@pytest.mark.parametrize("name", list(SPECS))
@pytest.mark.parametrize("cfl", [0.3, 20.0])
def test_advect_z_parity(torch, name, cfl):
    spec = SPECS[name]
    rng = np.random.default_rng(2)
    f = rng.random(spec.shape)
    tau = inputs.sweeps_dt_z(spec, cfl)
    ref = oracle.advect_z(spec, f, tau)
    for layout in (1, 2):
        s = _sldg(spec, layout)
        s.import_state(_dev(torch, f))
        s.advect_z(tau)
        got = s.export_state().cpu().numpy()
        s.check()
        assert _rel(got, ref) <= TOL
    s.advect_z(-0.37 * tau)
    ref2 = oracle.advect_z(spec, ref, -0.37 * tau)
    assert _rel(s.export_state().cpu().numpy(), ref2) <= TOL


@pytest.mark.parametrize("name", list(SPECS))
@pytest.mark.parametrize("cfl", [0.4, 2.5, 40.0])
def test_advect_v_parity(torch, name, cfl):
    spec = SPECS[name]
    rng = np.random.default_rng(3)
    f = rng.random(spec.shape)
    Ez = inputs.fourier_Ez(spec, seed=2, modes=3)
    tau = inputs.sweeps_dt_v(spec, Ez, cfl)
    ref = oracle.advect_v(spec, f, Ez, tau)
    for layout in (1, 2):
        s = _sldg(spec, layout)
        s.import_state(_dev(torch, f))
        s.set_Ez(_dev(torch, Ez))
        s.advect_v(tau)
        got = s.export_state().cpu().numpy()
        s.check()
        assert _rel(got, ref) <= TOL


@pytest.mark.parametrize("name", list(SPECS))
def test_advect_z_plane_kernel_is_bit_identical_to_the_column_walk(torch, monkeypatch, name):
    """Large Courant numbers (configs[2]: |CFL| = 20) send sldg_advect_z through the plane-tiled kernel (every z row read
    whole) instead of the per-column walk; same arithmetic, so the results must agree bit for bit."""
    spec = SPECS[name]
    rng = np.random.default_rng(17)
    f = rng.random(spec.shape)
    tau = 20.0 * spec.h[2] / max(abs(spec.lo[3]), abs(spec.hi[3]))
    outs = []
    for columns in (False, True):
        if columns:
            monkeypatch.setenv("SLDG_ADVECT_Z_COLUMNS", "1")
        else:
            monkeypatch.delenv("SLDG_ADVECT_Z_COLUMNS", raising=False)
        s = _sldg(spec)
        s.import_state(_dev(torch, f))
        n0 = s.launch_count()
        s.advect_z(tau)
        s.advect_z(-0.37 * tau)
        outs.append(s.export_state().cpu().numpy())
        s.check()
        s.close()
    assert np.array_equal(outs[0], outs[1])
    assert _rel(outs[0], oracle.advect_z(spec, oracle.advect_z(spec, f, tau), -0.37 * tau)) <= TOL


def test_integer_courant_numbers_are_bit_exact(torch):
    """A(0) = I, B(0) = 0: integer shifts copy the data with wrap, bit for bit (both sweeps)."""
    spec = GridSpec(n=(3, 2, 6, 8), order=(2, 2, 2, 1), lo=(0, 0, 0.0, -4.0), hi=(1, 1, 6.0, 4.0))
    rng = np.random.default_rng(4)
    f = rng.standard_normal(spec.shape)
    s = _sldg(spec)
    s.import_state(_dev(torch, f))
    s.advect_z(2.0)  # v nodes at -3.5..3.5, hz = 1: Courant numbers -7, -5, ..., 7
    got = s.export_state().cpu().numpy()
    v = spec.node_coords(3)
    Nz, Nv, Ny, Nx = spec.shape
    for V in range(Nv):
        k = int(round(v[V] * 2.0))
        ref = np.roll(f[:, V].reshape(6, 2, Ny, Nx), k, axis=0).reshape(Nz, Ny, Nx)
        assert np.array_equal(got[:, V], ref)
    # v sweep: Ez * tau / hv integer per line
    spec = GridSpec(n=(3, 2, 2, 8), order=(2, 2, 1, 2), lo=(0, 0, 0.0, -4.0), hi=(1, 1, 6.0, 4.0))
    f = rng.standard_normal(spec.shape)
    Nz, Nv, Ny, Nx = spec.shape
    k = rng.integers(-11, 12, size=(Nz, Ny, Nx))
    s = _sldg(spec)
    s.import_state(_dev(torch, f))
    s.set_Ez(_dev(torch, k.astype(np.float64)))
    s.advect_v(1.0)  # hv = 1
    got = s.export_state().cpu().numpy()
    s.check()
    for z in range(Nz):
        for y in range(Ny):
            for x in range(Nx):
                ref = np.roll(f[z, :, y, x].reshape(8, 2), k[z, y, x], axis=0).reshape(-1)
                assert np.array_equal(got[z, :, y, x], ref)


@pytest.mark.parametrize("name", list(SPECS))
def test_charge_density_and_mass_parity(torch, name):
    spec = SPECS[name]
    rng = np.random.default_rng(5)
    f = rng.random(spec.shape)
    s = _sldg(spec)
    s.import_state(_dev(torch, f))
    rho = s.charge_density().cpu().numpy()
    m = float(s.mass().cpu()[0])
    s.check()
    assert _rel(rho, oracle.charge_density(spec, f)) <= 1e-13
    assert abs(m - oracle.mass(spec, f)) <= 1e-13 * abs(m)


def _periodic_velocity(spec, seed, cfl, tau, Nz, wobble=0.12):
    """Bitwise-periodic smooth flow: a mean drift (sets the Courant number, so upstream cells land up to
    `cfl` cells away) plus a few low Fourier modes that deform them moderately (the upstream cells must
    stay convex: PAPER.md:190 'stability problems might appear if the approximated characteristics
    cross')."""
    nx, ny = spec.n[0], spec.n[1]
    rng = np.random.default_rng(seed)
    X, Y = np.meshgrid(np.arange(nx) / nx, np.arange(ny) / ny, indexing="xy")
    a = np.zeros((Nz, ny + 1, nx + 1))
    b = np.zeros_like(a)
    for z in range(Nz):
        ua = np.full((ny, nx), rng.uniform(-1, 1))
        ub = np.full((ny, nx), rng.uniform(-1, 1))
        for _ in range(4):
            kx, ky = rng.integers(0, 3, size=2)
            ua += wobble * rng.uniform(-1, 1) * np.cos(2 * np.pi * (kx * X + ky * Y) + rng.uniform(0, 6.28))
            ub += wobble * rng.uniform(-1, 1) * np.cos(2 * np.pi * (kx * X + ky * Y) + rng.uniform(0, 6.28))
        sc = cfl / max(np.abs(ua).max() * tau / spec.h[0], np.abs(ub).max() * tau / spec.h[1])
        for dst, src in ((a[z], ua), (b[z], ub)):
            dst[:ny, :nx] = sc * src
            dst[ny, :nx] = dst[0, :nx]
            dst[:, nx] = dst[:, 0]
    return a, b


@pytest.mark.parametrize("o", [2, 3])
@pytest.mark.parametrize("trace_order", [1, 2])
def test_xy_geometry_matches_oracle_coefficients(torch, o, trace_order):
    """Green's-theorem weights (GPU) vs clipped-polygon Gauss quadrature (oracle), block by block, plus the
    column-sum identity (mass conservation) evaluated on the GPU weights alone."""
    spec = GridSpec(n=(9, 7, 2, 3), order=(o, o, 1, 1), lo=(0, 0, 0, 0), hi=(1.8, 2.1, 1, 1))
    nx, ny = spec.n[0], spec.n[1]
    tau = 0.05
    a, b = _periodic_velocity(spec, 5, 0.9, tau, 2)
    s = _sldg(spec)
    s.import_state(_dev(torch, np.zeros(spec.shape)))
    s.set_vxy(_dev(torch, a), _dev(torch, b), 1)
    s.advect_xy(tau, trace_order)
    s.check()
    _, wg = oracle.gl(o)
    Wm = np.array([wg[m % o] * wg[m // o] for m in range(o * o)])
    for z in range(2):
        anchor, mask, W = (t.cpu().numpy() for t in s.debug_geometry(z))
        offs, er, es, eC = oracle.xy_plane_geometry(spec, a[z], b[z], tau, trace_order, 1)
        col = np.zeros((ny, nx, o * o))
        worst, scale = 0.0, 1.0
        for t in range(nx * ny):
            seen = 0
            for e in range(offs[t], offs[t + 1]):
                r, c = er[e] % nx, es[e] % ny
                dx, dy = (r - (t % nx + anchor[t, 0])) % nx, (c - (t // nx + anchor[t, 1])) % ny
                assert dx < 3 and dy < 3
                slot = dx + 3 * dy
                ref = (eC[e] / Wm[:, None]).T.reshape(-1)  # k-major [k][m]
                if (mask[t] >> slot) & 1:
                    seen |= 1 << slot
                    worst = max(worst, np.abs(W[t, slot] - ref).max())
                    scale = max(scale, np.abs(ref).max())
                    col[c, r] += (W[t, slot].reshape(o * o, o * o) * Wm[None, :]).sum(axis=1)
                else:
                    assert np.abs(ref).max() < 1e-13  # empty on the GPU <=> zero-area piece
            assert seen == mask[t]
        # Green boundary integrals lose ~1e-16 absolute per O(1) edge term; times the adjoint coefficients and
        # 1/W_m (up to 13 at o=3) this is a few 1e-12 per block at o=3, ~1e-14 at o=2 (tolerances)
        assert worst < (1e-13 if o == 2 else 5e-12) * scale, (worst, scale)
        assert np.abs(col - Wm).max() < 5e-14


@pytest.mark.parametrize("o,ncell", [(2, 128), (3, 96)])
def test_geometry_column_sums_at_bench_size(torch, o, ncell):
    """Property that holds at any size (mass conservation, SURVEY.md 8(c)-2 pin (i)): on the ITG field of
    the headline config (full nx x ny plane, a few z nodes) every source DOF's weights sum to W_k.  The ITG
    field decays to ~1e-18 away from the annulus, which produces upstream cells whose corners sit within
    rounding of grid lines (zero-area slivers) -- the degenerate cases of the clipping."""
    spec = inputs.itg_grid(ncell, ncell, 2, 1, o)
    a, b, _, _ = inputs.itg_fields(spec, 4.0, 0.8)
    s = _sldg(spec)
    s.import_state(_dev(torch, np.zeros(spec.shape)))
    s.set_vxy(_dev(torch, a), _dev(torch, b), 1)
    s.advect_xy(4.0, 2)
    s.check()
    _, wg = oracle.gl(o)
    Wm = torch.tensor([wg[m % o] * wg[m // o] for m in range(o * o)], dtype=torch.float64, device="cuda")
    nx = ny = ncell
    t = torch.arange(nx * ny, device="cuda")
    ti, tj = t % nx, t // nx
    for z in range(spec.shape[0]):
        anchor, mask, W = s.debug_geometry(z)
        anchor, mask = anchor.long(), mask.long()
        col = torch.zeros(ny * nx, o * o, dtype=torch.float64, device="cuda")
        for slot in range(9):
            on = ((mask >> slot) & 1).bool()
            r = (ti + anchor[:, 0] + slot % 3) % nx
            c = (tj + anchor[:, 1] + slot // 3) % ny
            w = W[on, slot].reshape(-1, o * o, o * o) * Wm[None, None, :]  # [k][m]
            col.index_add_(0, (c * nx + r)[on], w.sum(dim=2))
        assert float((col - Wm[None, :]).abs().max()) < 5e-14


def _xy_case(torch, spec, f, a, b, tau, trace_order, periodic, steps=1):
    s = _sldg(spec)
    s.import_state(_dev(torch, f))
    s.set_vxy(_dev(torch, a), _dev(torch, b), periodic)
    ref = f
    for _ in range(steps):
        s.advect_xy(tau, trace_order)
        ref = oracle.advect_xy(spec, ref, a, b, tau, trace_order, periodic)
    got = s.export_state().cpu().numpy()
    s.check()
    return got, ref, s


@pytest.mark.parametrize("o", [2, 3])
@pytest.mark.parametrize("trace_order", [1, 2])
@pytest.mark.parametrize("cfl", [0.5, 1.7])
def test_advect_xy_parity_random_periodic_flow(torch, o, trace_order, cfl):
    spec = GridSpec(n=(11, 9, 3, 13), order=(o, o, 1, 2), lo=(0, 0, 0, 0), hi=(2.2, 1.8, 1, 1))
    rng = np.random.default_rng(6)
    f = rng.random(spec.shape)
    tau = 0.1
    a, b = _periodic_velocity(spec, 8, cfl, tau, spec.shape[0])
    got, ref, s = _xy_case(torch, spec, f, a, b, tau, trace_order, 1, steps=2)
    assert _rel(got, ref) <= TOL
    m0, m1 = oracle.mass(spec, f), float(s.mass().cpu()[0])
    assert abs(m1 - m0) <= 1e-13 * abs(m0)


@pytest.mark.parametrize("o", [2, 3])
def test_advect_xy_parity_rotation_and_swirl(torch, o):
    """Config 1 shapes at a size the oracle finishes in seconds: 48x48 cells, 40 planes."""
    spec = inputs.bumps_grid(48, 40, o)
    f = inputs.bumps_initial_f(spec, seed=1)
    a, b = inputs.rotation_velocity(spec)
    got, ref, _ = _xy_case(torch, spec, f, a, b, 2 * math.pi / 40, 2, 0, steps=3)
    assert _rel(got, ref) <= TOL
    tau = 0.05
    a, b = inputs.swirl_velocity(spec, 0.5 * tau)
    got, ref, s = _xy_case(torch, spec, f, a, b, tau, 2, 1, steps=2)
    assert _rel(got, ref) <= TOL
    m0, m1 = oracle.mass(spec, f), float(s.mass().cpu()[0])
    assert abs(m1 - m0) <= 1e-13 * abs(m0)


def test_advect_xy_mixed_streaming_and_direct_blocks(torch):
    """o = 2: the blocks (strip x segment) whose anchors vary too much for the streaming kernel's ring go to the
    direct kernel, the others stream -- decided on the device.  A flow whose y displacement swings by +-2.5 cells
    inside the first segment of 128 rows and is nearly uniform in the second must use both kernels in one step."""
    spec = GridSpec(n=(16, 160, 1, 24), order=(2, 2, 1, 1), lo=(0.0, 0.0, 0.0, 0.0), hi=(1.0, 10.0, 1.0, 1.0))
    rng = np.random.default_rng(21)
    f = rng.random(spec.shape)
    tau = 1.0
    yv = np.linspace(0.0, 1.0, spec.n[1] + 1)  # y / Ly at the vertices
    xv = np.linspace(0.0, 1.0, spec.n[0] + 1)
    env = (0.5 + 0.5 * np.cos(2 * np.pi * (yv - 0.4))) ** 4
    by = (2.5 * np.sin(2 * np.pi * (yv - 0.4)) * env + 0.3) * spec.h[1] / tau
    ax = 0.4 * np.sin(2 * np.pi * xv) * spec.h[0] / tau
    a = np.ascontiguousarray(np.broadcast_to(ax[None, None, :], (1, spec.n[1] + 1, spec.n[0] + 1)))
    b = np.ascontiguousarray(np.broadcast_to(by[None, :, None], (1, spec.n[1] + 1, spec.n[0] + 1)))
    for u in (a, b):  # bitwise periodic
        u[:, -1, :] = u[:, 0, :]
        u[:, :, -1] = u[:, :, 0]
    got, ref, s = _xy_case(torch, spec, f, a, b, tau, 2, 1)
    direct_blocks = s.debug_counter(0)
    assert 0 < direct_blocks < 2 * 2, direct_blocks  # 2 strips x 2 segments x 1 z node
    assert _rel(got, ref) <= TOL
    m0 = oracle.mass(spec, f)
    assert abs(float(s.mass().cpu()[0]) - m0) <= 1e-13 * m0


def test_zero_and_constant_velocity(torch):
    spec = GridSpec(n=(6, 5, 1, 4), order=(2, 2, 1, 2), lo=(0, 0, 0, 0), hi=(3.0, 2.5, 1, 1))
    rng = np.random.default_rng(9)
    f = rng.standard_normal(spec.shape)
    z = np.zeros((1, 6, 7))
    got, ref, _ = _xy_case(torch, spec, f, z, z, 0.3, 2, 1)
    assert np.abs(got - f).max() < 1e-14
    # integer Courant numbers in x and y: pure roll of cells (to round-off)
    a = np.full((1, 6, 7), 2 * spec.h[0])
    b = np.full((1, 6, 7), -1 * spec.h[1])
    got, ref, _ = _xy_case(torch, spec, f, a, b, 1.0, 1, 1)
    Nz, Nv, Ny, Nx = spec.shape
    roll = np.roll(np.roll(f.reshape(Nz, Nv, 5, 2, 6, 2), 2, axis=4), -1, axis=2).reshape(spec.shape)
    assert np.abs(got - roll).max() < 1e-13
    assert _rel(got, ref) <= TOL


def test_config0_tiny_itg_20_strang_steps(torch):
    """BASELINE.json configs[0]: 16x16x8x16 cells, o=2, dt=2, 20 Strang steps; parity and mass."""
    spec = inputs.itg_grid(16, 16, 8, 16, 2)
    f = inputs.itg_initial_f(spec)
    dt = 2.0
    a, b, Ez, _ = inputs.itg_fields(spec, dt, 0.8)
    s = _sldg(spec)
    s.import_state(_dev(torch, f))
    s.set_Ez(_dev(torch, Ez))
    s.set_vxy(_dev(torch, a), _dev(torch, b), 1)
    ref = f.copy()
    m0 = oracle.mass(spec, f)
    assert abs(float(s.mass().cpu()[0]) - m0) <= 1e-14 * m0
    for n in range(20):
        s.strang_step(dt)
        oracle.strang_step(spec, ref, Ez, a, b, dt, 2, 1)
        m = float(s.mass().cpu()[0])
        assert abs(m - m0) <= 1e-13 * m0, (n, m, m0)
    got = s.export_state().cpu().numpy()
    s.check()
    assert _rel(got, ref) <= TOL
    rho = s.charge_density().cpu().numpy()
    assert _rel(rho, oracle.charge_density(spec, ref)) <= TOL
    ms = s.last_timing_ms()
    fused = (int(ms[6]) & 6) == 6
    timed = [ms[0], ms[2], ms[3], ms[4]] if fused else ms[:6]
    assert all(t > 0 for t in timed) and ms[7] >= max(ms[:6])
    assert s.launch_count() >= 20 * (4 if fused else 6)


@pytest.mark.gpu
@pytest.mark.parametrize("o,cells", [(2, (6, 5, 8, 16)), (2, (4, 4, 16, 64)), (3, (4, 3, 6, 16)), (2, (3, 3, 5, 7))])
@pytest.mark.parametrize("cfl", [0.4, 7.3])
def test_fused_sweep_pairs_are_bit_identical_to_separate_sweeps(torch, monkeypatch, o, cells, cfl):
    """sldg_strang_step runs z,v and v,z as one kernel each where the (z,v) plane fits in shared memory: the
    state must equal, bit for bit, the one produced by the five separate substep calls, for small and large
    Courant numbers (wrap-around of the rotated columns) and ragged sizes."""
    spec = inputs.itg_grid(*cells, o)
    rng = np.random.default_rng(7)
    f = rng.random(spec.shape)
    dt = 2.0
    a, b, Ez, _ = inputs.itg_fields(spec, dt, 0.6)
    Ez = Ez * (cfl * spec.h[3] / (0.5 * dt) / max(np.abs(Ez).max(), 1e-300))
    dtz = dt  # z Courant numbers come from the v nodes themselves (up to |v| dt/2 / h_z)
    outs = []
    for fuse in (True, False):
        if fuse:
            monkeypatch.delenv("SLDG_NO_FUSE", raising=False)
        else:
            monkeypatch.setenv("SLDG_NO_FUSE", "1")
        s = _sldg(spec)
        s.import_state(_dev(torch, f))
        s.set_Ez(_dev(torch, Ez))
        s.set_vxy(_dev(torch, a), _dev(torch, b), 1)
        if fuse:
            for _ in range(2):
                s.strang_step(dtz)
            assert (int(s.last_timing_ms()[6]) & 6) == 6, "the fused path did not run"
        else:
            for _ in range(2):
                s.advect_z(0.5 * dtz)
                s.advect_v(0.5 * dtz)
                s.advect_xy(dtz, 2)
                s.advect_v(0.5 * dtz)
                s.advect_z(0.5 * dtz)
        s.check()
        outs.append(s.export_state().cpu().numpy())
        s.close()
    assert np.array_equal(outs[0], outs[1])


def test_mass_drift_over_200_strang_steps(torch):
    """BASELINE.json configs[3] runs 200 Strang steps and records the mass drift every step: it must stay below
    1e-13 relative over the whole run.  (Before the conservation correction of the 1d overlap matrices -- see
    eval_shift -- every sweep lost 1.5e-16 with a fixed sign and 200 steps ended at 1.5e-13.)"""
    spec = inputs.itg_grid(64, 64, 4, 16, 2)  # configs[3]'s resolution in (x, y), fewer z and v cells
    dt = 4.0
    a, b, Ez, _ = inputs.itg_fields(spec, dt, 0.8)
    s = _sldg(spec)
    s.import_state(_dev(torch, inputs.itg_initial_f(spec)))
    s.set_Ez(_dev(torch, Ez))
    s.set_vxy(_dev(torch, a), _dev(torch, b), 1)
    m0 = float(s.mass().cpu()[0])
    worst = 0.0
    for n in range(200):
        s.strang_step(dt)
        if n % 10 == 9:
            worst = max(worst, abs(float(s.mass().cpu()[0]) - m0) / abs(m0))
    s.check()
    assert worst <= 1e-13, worst


def test_layouts_agree_bitwise_on_a_strang_step(torch):
    spec = inputs.itg_grid(8, 8, 4, 8, 2)
    f = inputs.itg_initial_f(spec)
    a, b, Ez, _ = inputs.itg_fields(spec, 2.0, 0.8)
    outs = []
    for layout in (1, 2, 3):
        s = _sldg(spec, layout)
        s.import_state(_dev(torch, f))
        s.set_Ez(_dev(torch, Ez))
        s.set_vxy(_dev(torch, a), _dev(torch, b), 1)
        s.strang_step(2.0)
        outs.append(s.export_state().cpu().numpy())
        s.check()
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


def test_strang_step_host_entry_point(torch):
    spec = inputs.itg_grid(8, 8, 4, 8, 2)
    f = inputs.itg_initial_f(spec)
    a, b, Ez, _ = inputs.itg_fields(spec, 2.0, 0.8)
    s = _sldg(spec)
    s.import_state_host(f)
    rho = np.empty((spec.shape[0], spec.shape[2], spec.shape[3]))
    mass = np.empty(1)
    s.strang_step_host(2.0, Ez, a, b, 1, rho, mass)
    ref = oracle.strang_step(spec, f.copy(), Ez, a, b, 2.0, 2, 1)
    assert _rel(rho, oracle.charge_density(spec, ref)) <= TOL
    assert abs(mass[0] - oracle.mass(spec, ref)) <= 1e-13 * abs(mass[0])
    out = np.empty_like(f)
    s.export_state_host(out)
    assert _rel(out, ref) <= TOL


def test_geometry_error_words(torch):
    from paper_2212_03036_b200.binding import SLDG_ESTENCIL, SldgError
    spec = GridSpec(n=(8, 8, 1, 2), order=(2, 2, 1, 1), lo=(0, 0, 0, 0), hi=(1, 1, 1, 1))
    s = _sldg(spec)
    s.import_state(_dev(torch, np.zeros(spec.shape)))
    # a shear so strong that upstream cells span more than three source cells
    a = np.zeros((1, 9, 9))
    a[0] = (np.arange(9)[:, None] * 5.0) * spec.h[0]
    s.set_vxy(_dev(torch, a), _dev(torch, np.zeros((1, 9, 9))), 0)
    s.advect_xy(1.0, 1)
    with pytest.raises(SldgError) as ei:
        s.check()
    assert ei.value.code == SLDG_ESTENCIL
    s.check()  # cleared


def test_geometry_error_egeom_both_ways(torch):
    """SLDG_EGEOM, provoked both ways, and the oracle raises on the same
    input: (i) crossed characteristics -- a field converging so strongly that Euler's foot map (1 - tau k) x flips the
    orientation of every upstream cell; (ii) a singular Vandermonde system -- one Euler step of the solid rotation
    with tau = 1 turns the Q^1 node feet by 45 degrees onto the axes through their centre, where the monomial xy
    vanishes at all four of them.  A slightly smaller step (tau = 0.9) is fine on both sides."""
    from paper_2212_03036_b200.binding import SLDG_EGEOM, SldgError
    spec = GridSpec(n=(8, 8, 1, 2), order=(2, 2, 1, 1), lo=(-1, -1, 0, 0), hi=(1, 1, 1, 1))
    XV, YV = np.meshgrid(spec.vertex_coords(0), spec.vertex_coords(1), indexing="xy")
    rng = np.random.default_rng(13)
    f = rng.random(spec.shape)
    cases = [((1.5 * XV)[None], np.zeros((1, 9, 9)), 1.0), ((-YV)[None], XV[None].copy(), 1.0)]
    for a, b, tau in cases:
        with pytest.raises(oracle.OracleError):
            oracle.advect_xy(spec, f, a, b, tau, 1, 0)
        s = _sldg(spec)
        s.import_state(_dev(torch, f))
        s.set_vxy(_dev(torch, a), _dev(torch, b), 0)
        s.advect_xy(tau, 1)
        with pytest.raises(SldgError) as ei:
            s.check()
        assert ei.value.code == SLDG_EGEOM
        s.check()  # cleared
        s.close()
    a, b, _ = cases[1]
    s = _sldg(spec)
    s.import_state(_dev(torch, f))
    s.set_vxy(_dev(torch, a), _dev(torch, b), 0)
    s.advect_xy(0.9, 1)
    s.check()
    assert _rel(s.export_state().cpu().numpy(), oracle.advect_xy(spec, f, a, b, 0.9, 1, 0)) <= TOL
    s.close()


@pytest.mark.parametrize("o,cells", [(2, (6, 5, 8, 16)), (2, (4, 4, 40, 64)), (3, (4, 3, 19, 16)), (2, (3, 3, 17, 7)),
                                     (1, (5, 4, 33, 20)), (2, (4, 4, 20, 128)), (2, (4, 5, 16, 100))])
@pytest.mark.parametrize("zcfl", [0.3, 1.7])
def test_z_tiled_sweep_pairs_are_bit_identical_to_separate_sweeps(torch, monkeypatch, o, cells, zcfl):
    """The z-tiled pair kernel (sldg_tiled_sweeps.cu: planes that do not fit in shared memory, small z Courant numbers)
    against the five separate substep calls, bit for bit: tiles with a ragged last tile, halos that wrap around the
    periodic z axis, odd cell counts, v shifts of several cells, 128 v cells (the paper's grid)."""
    spec = inputs.itg_grid(*cells, o)
    rng = np.random.default_rng(11)
    f = rng.random(spec.shape)
    dt = 2.0 * zcfl * spec.h[2] / inputs.ITG_VMAX        # max |v| dt/2 / h_z = zcfl
    a, b, Ez, _ = inputs.itg_fields(spec, dt, 0.5)
    Ez = Ez * (2.3 * spec.h[3] / (0.5 * dt) / max(np.abs(Ez).max(), 1e-300))
    outs = []
    for tiled in (True, False):
        if tiled:
            monkeypatch.delenv("SLDG_NO_FUSE", raising=False)
            monkeypatch.setenv("SLDG_FORCE_TILE", "1")
        else:
            monkeypatch.delenv("SLDG_FORCE_TILE", raising=False)
            monkeypatch.setenv("SLDG_NO_FUSE", "1")
        s = _sldg(spec)
        s.import_state(_dev(torch, f))
        s.set_Ez(_dev(torch, Ez))
        s.set_vxy(_dev(torch, a), _dev(torch, b), 1)
        launches0 = s.launch_count()
        if tiled:
            for _ in range(2):
                s.strang_step(dt)
            assert (int(s.last_timing_ms()[6]) & 6) == 6, "the pairs did not run fused"
            # 2 steps x (pair, geometry, scan, stream/direct apply..., pair): the pairs are ONE launch each
            assert s.launch_count() - launches0 <= 2 * 6
        else:
            for _ in range(2):
                s.advect_z(0.5 * dt)
                s.advect_v(0.5 * dt)
                s.advect_xy(dt, 2)
                s.advect_v(0.5 * dt)
                s.advect_z(0.5 * dt)
        s.check()
        outs.append(s.export_state().cpu().numpy())
        s.close()
    assert np.array_equal(outs[0], outs[1])


def test_timing_history_matches_last_timing(torch):
    """sldg_timing_history returns, for each of the last n Strang steps, what sldg_last_timing_ms returned right after
    that step; single substep calls in between do not disturb the recorded steps."""
    spec = inputs.itg_grid(12, 10, 6, 16, 2)
    f = inputs.itg_initial_f(spec)
    a, b, Ez, _ = inputs.itg_fields(spec, 2.0, 0.8)
    s = _sldg(spec)
    s.import_state(_dev(torch, f))
    s.set_Ez(_dev(torch, Ez))
    s.set_vxy(_dev(torch, a), _dev(torch, b), 1)
    want = []
    for n in range(5):
        s.strang_step(2.0)
        want.append(s.last_timing_ms())
        if n == 2:
            s.advect_z(0.1)
            s.advect_xy(0.1, 2)
    got = s.timing_history(5)
    assert np.allclose(np.array(got), np.array(want), rtol=0, atol=0)
    assert all(g[7] > 0 and abs(g[7] - (g[0] + g[1] + g[3] + g[4] + g[5])) < 0.05 for g in got)
    s.close()


@pytest.mark.parametrize("no_fuse", [False, True])
@pytest.mark.parametrize("cells", [(6, 7, 5, 12), (6, 7, 5, 16), (5, 9, 7, 64), (4, 8, 3, 96)])
def test_strang_step_host_overlapped_transfers(torch, monkeypatch, no_fuse, cells):
    """sldg_strang_step_host uploads E_z in chunks of y rows under the fused z,v pair, which is then launched chunk by
    chunk: same bits of the state as the device-resident step with the fields set beforehand -- two steps with different
    fields, a number of y rows that the chunks do not divide, and with the fused pairs switched off (one plain upload).
    Where the v lines are whole warps without padding (16 and 64 v cells at o = 2) the v,z pair also forms the charge density
    from its own results and is launched chunk by chunk with the downloads in between: rho against the reduction kernel
    (the order of the v sum differs) and against the oracle."""
    if no_fuse:
        monkeypatch.setenv("SLDG_NO_FUSE", "1")
    spec = inputs.itg_grid(*cells, 2)
    f = inputs.itg_initial_f(spec, eps=0.05)
    dt = 2.0
    fields = [inputs.itg_fields(spec, dt, 0.8)[:3], inputs.itg_fields(spec, dt, 0.5)[:3]]
    fields[1] = tuple(np.ascontiguousarray(-x) for x in fields[1])
    outs = []
    for host in (False, True):
        s = _sldg(spec)
        s.import_state(_dev(torch, f))
        rho = np.full((spec.shape[0], spec.shape[2], spec.shape[3]), np.nan)
        mass = np.empty(1)
        for a, b, Ez in fields:
            if host:
                rho[...] = np.nan
                s.strang_step_host(dt, Ez, a, b, 1, rho, mass)
            else:
                s.set_Ez(_dev(torch, Ez))
                s.set_vxy(_dev(torch, a), _dev(torch, b), 1)
                s.strang_step(dt)
        s.check()
        outs.append(s.export_state().cpu().numpy())
        if host:
            ref = s.charge_density().cpu().numpy()
            assert np.abs(rho - ref).max() <= 1e-14 * np.abs(ref).max()
            assert _rel(rho, oracle.charge_density(spec, outs[-1])) <= 1e-13
            assert abs(mass[0] - float(s.mass().cpu()[0])) <= 1e-14 * abs(mass[0])
        s.close()
    assert np.array_equal(outs[0], outs[1])

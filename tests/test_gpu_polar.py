"""GPU parity of the polar delta-g step: source term, theta-only periodic
tracing, Algorithm 1 steps 2-4, 6-9 with prescribed fields, against oracle/polar.py through the C-ABI."""
import numpy as np
import pytest

import oracle
from oracle import polar
from paper_2212_03036_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1e-11


@pytest.fixture(scope="module")
def torch():
    import torch as t
    if not t.cuda.is_available():
        pytest.skip("needs a CUDA device")
    return t


def _ctx(torch, spec, f, fl, dv, dr, layout=0):
    from paper_2212_03036_b200.binding import Sldg
    s = Sldg(spec, layout=layout)
    cu = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
    s.import_state(cu(f))
    s.set_Ez(cu(fl["Ez"]))
    s.set_vxy(cu(fl["a"]), cu(fl["b"]), 2)
    s.set_equilibrium(cu(dv), cu(dr))
    s.set_source_fields(cu(fl["dz_phi"]), cu(fl["dth_phi"]))
    return s


@pytest.mark.parametrize("o,cells", [(2, (6, 8, 3, 8)), (3, (5, 4, 2, 7)), (1, (7, 6, 4, 16))])
@pytest.mark.parametrize("layout", [1, 2])
def test_source_step_parity(torch, o, cells, layout):
    spec = inputs.polar_grid(*cells, o)
    _, dv, dr = inputs.polar_equilibrium(spec)
    fl = inputs.polar_fields(spec, 4.0)
    f = inputs.polar_initial_dg(spec, eps=0.1)
    s = _ctx(torch, spec, f, fl, dv, dr, layout)
    s.source_step(0.7)
    s.source_step(-0.2)
    got = s.export_state().cpu().numpy()
    want = polar.source_step(polar.source_step(f, fl["dz_phi"], fl["dth_phi"], dv, dr, 0.7), fl["dz_phi"], fl["dth_phi"], dv, dr, -0.2)
    assert np.abs(got - want).max() <= 1e-14 * np.abs(want).max()
    s.close()


@pytest.mark.parametrize("o,cells,cfl", [(2, (16, 24, 4, 16), 0.8), (3, (8, 12, 2, 8), 0.5)])
def test_polar_strang_step_with_sources_parity_and_mass(torch, o, cells, cfl):
    # (o = 3 on this coarse 8 x 12 mesh: at a Courant number of 0.8 the sheared flow near r_min makes the data itself
    # grow fourfold per step, measured on both sides, and the difference with it; 0.5 is resolved)
    spec = inputs.polar_grid(*cells, o)
    _, dv, dr = inputs.polar_equilibrium(spec)
    dt = 4.0
    fl = inputs.polar_fields(spec, dt, cfl)
    f = inputs.polar_initial_dg(spec, eps=0.1)
    s = _ctx(torch, spec, f, fl, dv, dr)
    ref = f.copy()
    for n in range(5):
        s.strang_step_sources(dt)
        ref = polar.strang_step_sources(spec, np.ascontiguousarray(ref), fl, dv, dr, dt)
    s.check()
    got = s.export_state().cpu().numpy()
    assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()
    scale = oracle.mass(spec, np.abs(ref))
    assert abs(float(s.mass().cpu()[0]) - oracle.mass(spec, f)) <= 1e-13 * scale
    s.close()


def test_data_at_the_radial_ends_stays_there(torch):
    # the periodic wrap of the 2d kernels along axis 0 is never exercised when the radial velocity vanishes at the ends
    spec = inputs.polar_grid(16, 16, 2, 8, 2)
    _, dv, dr = inputs.polar_equilibrium(spec)
    dt = 4.0
    fl = inputs.polar_fields(spec, dt, 0.8)
    f = np.zeros(spec.shape)
    f[:, :, :, :2] = 1.0
    f[:, :, :, -2:] = 2.0
    f *= (1.0 + 0.3 * np.cos(spec.node_coords(1)))[None, None, :, None]
    s = _ctx(torch, spec, f, fl, 0.0 * dv, 0.0 * dr)
    ref = f.copy()
    for n in range(3):
        s.strang_step_sources(dt)
        ref = polar.strang_step_sources(spec, np.ascontiguousarray(ref), fl, 0.0 * dv, 0.0 * dr, dt)
    s.check()
    got = s.export_state().cpu().numpy()
    assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()
    half = spec.N[0] // 2
    inner = got.copy()
    inner[:, :, :, half:] = 0.0
    inner0 = f.copy()
    inner0[:, :, :, half:] = 0.0
    assert abs(oracle.mass(spec, inner) - oracle.mass(spec, inner0)) <= 1e-12 * oracle.mass(spec, f)
    s.close()


def _polar_ctx(torch, spec, dg):
    from paper_2212_03036_b200.binding import Sldg
    cu = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
    rv = spec.vertex_coords(0)
    n0, dln_n0, T, _ = inputs.polar_profiles(rv)
    _, dv, dr = inputs.polar_equilibrium(spec)
    s = Sldg(spec)
    s.import_state(cu(dg))
    s.set_polar_profiles(cu(rv * n0), cu(dln_n0), cu(T))
    s.set_equilibrium(cu(dv), cu(dr))
    return s, n0, dln_n0, T, dv, dr


@pytest.mark.parametrize("o,cells", [(2, (16, 24, 4, 16)), (3, (8, 12, 2, 8)), (1, (9, 12, 5, 12)), (2, (20, 15, 3, 8))])
def test_polar_quasi_neutrality_solve_matches_the_oracle(torch, o, cells):
    # eq. (2) as printed: Fourier sums in theta and z, tridiagonal solves in r (Neumann / Dirichlet), drift with zero
    # radial ends -- a direct solver on both sides, so the potential agrees to round-off
    spec = inputs.polar_grid(*cells, o)
    dg = inputs.polar_initial_dg(spec, eps=0.1)
    s, n0, dln_n0, T, dv, dr = _polar_ctx(torch, spec, dg)
    s.polar_field_step()
    want = polar.polar_field_step(spec, dg, n0, dln_n0, T)
    phi = s.get_polar_phi().cpu().numpy()
    scale = np.abs(want["phi"]).max()
    assert np.abs(phi - want["phi"]).max() <= 1e-11 * scale
    Ez, a, b = (x.cpu().numpy() for x in s.get_fields())
    dz, dth = (x.cpu().numpy() for x in s.get_source_fields())
    assert np.abs(a - want["a"]).max() <= 1e-10 * np.abs(want["a"]).max()
    assert np.abs(b - want["b"]).max() <= 1e-10 * np.abs(want["b"]).max()
    assert np.abs(Ez - want["Ez"]).max() <= 1e-10 * np.abs(want["Ez"]).max()
    assert np.abs(dz - want["dz_phi"]).max() <= 1e-10 * np.abs(want["Ez"]).max()
    assert np.abs(dth - want["dth_phi"]).max() <= 1e-10 * np.abs(want["dth_phi"]).max()
    assert np.all(a[:, :, 0] == 0.0) and np.all(a[:, :, -1] == 0.0)
    assert np.array_equal(a[:, -1], a[:, 0]) and np.array_equal(b[:, -1], b[:, 0])
    s.close()


@pytest.mark.parametrize("o,cells,eps", [(2, (16, 24, 4, 16), 1e-6), (2, (16, 24, 4, 16), 0.05), (3, (8, 12, 2, 8), 0.02)])
def test_polar_algorithm1_self_consistent_steps(torch, o, cells, eps):
    # the paper's own set-up on a small mesh: Algorithm 1 with all nine steps, potential from eq. (2)
    spec = inputs.polar_grid(*cells, o)
    dg = inputs.polar_initial_dg(spec, eps=eps)
    s, n0, dln_n0, T, dv, dr = _polar_ctx(torch, spec, dg)
    ref = dg.copy()
    dt = 4.0
    for n in range(4):
        s.step_algorithm1_polar(dt)
        ref, fs = polar.polar_algorithm1_step(spec, ref, n0, dln_n0, T, dv, dr, dt)
    s.check()
    got = s.export_state().cpu().numpy()
    assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()
    scale = oracle.mass(spec, np.abs(ref))
    assert abs(float(s.mass().cpu()[0]) - oracle.mass(spec, dg)) <= 1e-13 * scale
    s.close()


@pytest.mark.parametrize("fuse", [True, False])
@pytest.mark.parametrize("o,cells,eps", [(2, (16, 24, 4, 16), 0.05), (3, (8, 12, 2, 8), 0.02)])
def test_polar_algorithm2_predictor_corrector(torch, monkeypatch, fuse, o, cells, eps):
    # Algorithm 2 with all thirteen steps: the predictor's source step is out of place, the three buffers rotate
    if not fuse:
        monkeypatch.setenv("SLDG_NO_FUSE", "1")
    spec = inputs.polar_grid(*cells, o)
    dg = inputs.polar_initial_dg(spec, eps=eps)
    s, n0, dln_n0, T, dv, dr = _polar_ctx(torch, spec, dg)
    ref = dg.copy()
    dt = 4.0
    for n in range(3):
        s.step_algorithm2_polar(dt)
        ref, fs = polar.polar_algorithm2_step(spec, ref, n0, dln_n0, T, dv, dr, dt)
        got = s.export_state().cpu().numpy()
        assert np.abs(got - ref).max() <= TOL * np.abs(ref).max(), n
    s.check()
    scale = oracle.mass(spec, np.abs(ref))
    assert abs(float(s.mass().cpu()[0]) - oracle.mass(spec, dg)) <= 1e-13 * scale
    s.close()

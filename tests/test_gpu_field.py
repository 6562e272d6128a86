"""GPU parity of the field step, the invariants and Algorithms 1 and 2 against
oracle/field.py, through the C-ABI.  The potential comes from an iterative solver: its bar is kappa * tol relative to
max |phi|; the state after whole time steps keeps the 1e-11 bar of north_star."""
import numpy as np
import pytest

import oracle
from oracle import field
from paper_2212_03036_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1e-11


@pytest.fixture(scope="module")
def torch():
    import torch as t
    if not t.cuda.is_available():
        pytest.skip("needs a CUDA device")
    return t


def _ctx(torch, spec, f, B=1.0):
    from paper_2212_03036_b200.binding import Sldg
    s = Sldg(spec)
    s.import_state(torch.from_numpy(f).cuda())
    n0, Te = inputs.itg_vertex_profiles(spec)
    s.set_profiles(torch.from_numpy(n0).cuda(), torch.from_numpy(Te).cuda(), B)
    return s, n0, Te


def _rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


@pytest.mark.parametrize("o,cells", [(2, (16, 16, 8, 16)), (3, (9, 7, 3, 8)), (1, (12, 10, 5, 16)), (2, (40, 36, 2, 8))])
@pytest.mark.parametrize("eps", [1e-6, 0.2])
def test_field_step_matches_the_oracle(torch, o, cells, eps):
    spec = inputs.itg_grid(*cells, o)
    f = inputs.itg_initial_f(spec, eps=eps)
    s, n0, Te = _ctx(torch, spec, f, B=1.3)
    s.field_step(1e-14, 5000)
    iters, relres = s.field_info()
    assert relres <= 1e-13, (iters, relres)
    want = field.field_step(spec, oracle.charge_density(spec, f), n0, Te, 1.3)
    phi = s.get_phi().cpu().numpy()
    Ez, a, b = (x.cpu().numpy() for x in s.get_fields())
    assert _rel(phi, want["phi"]) <= 1e-9
    scale = np.abs(want["phi"]).max()
    assert np.abs(a - want["a"]).max() <= 1e-9 * scale / spec.h[1]
    assert np.abs(b - want["b"]).max() <= 1e-9 * scale / spec.h[0]
    assert np.abs(Ez - want["Ez"]).max() <= 1e-9 * scale / (spec.h[2] / o)
    assert np.array_equal(a[:, -1, :], a[:, 0, :]) and np.array_equal(a[:, :, -1], a[:, :, 0])  # bitwise periodic
    assert np.array_equal(b[:, -1, :], b[:, 0, :]) and np.array_equal(b[:, :, -1], b[:, :, 0])
    d = s.diagnostics(inputs.ITG_RP)
    dw = field.diagnostics(spec, f, want["phi"], want["phi_nodes"], inputs.ITG_RP)
    for k in ("mass", "l2", "kinetic"):
        assert abs(d[k] - dw[k]) <= 1e-12 * abs(dw[k]), k
    assert abs(d["electric"] - dw["electric"]) <= 1e-9 * dw["electric"]
    assert abs(d["potential"] - dw["potential"]) <= 1e-9 * scale * dw["mass"]
    s.close()


def test_config0_self_consistent_algorithm1_20_steps(torch):
    # BASELINE.json configs[0] with the potential from the quasi-neutrality solve instead of the prescribed one
    spec = inputs.itg_grid(16, 16, 8, 16, 2)
    f = inputs.itg_initial_f(spec)
    s, n0, Te = _ctx(torch, spec, f)
    ref = f.copy()
    m0 = oracle.mass(spec, f)
    for n in range(20):
        s.step_algorithm1(2.0, 1e-14, 5000)
        ref, fs = field.algorithm1_step(spec, ref, n0, Te, 2.0)
        if n in (0, 9, 19):
            got = s.export_state().cpu().numpy()
            assert _rel(got, ref) <= TOL, n
            assert abs(float(s.mass().cpu()[0]) - m0) <= 1e-13 * m0
    s.check()
    s.close()


@pytest.mark.parametrize("fuse", [True, False])
@pytest.mark.parametrize("o,cells,eps", [(2, (12, 10, 4, 16), 0.05), (3, (8, 8, 2, 8), 0.05)])
def test_algorithm2_predictor_corrector_matches_the_oracle(torch, monkeypatch, fuse, o, cells, eps):
    if not fuse:
        monkeypatch.setenv("SLDG_NO_FUSE", "1")
    spec = inputs.itg_grid(*cells, o)
    f = inputs.itg_initial_f(spec, eps=eps)
    s, n0, Te = _ctx(torch, spec, f)
    ref = f.copy()
    m0 = oracle.mass(spec, f)
    for n in range(4):
        s.step_algorithm2(4.0, 1e-14, 5000)
        ref, fs = field.algorithm2_step(spec, ref, n0, Te, 4.0)
        got = s.export_state().cpu().numpy()
        assert _rel(got, ref) <= TOL, n
    assert abs(float(s.mass().cpu()[0]) - m0) <= 1e-13 * m0
    # the fields left in the context are those of the corrector (phi^{n+1/2})
    Ez, a, b = (x.cpu().numpy() for x in s.get_fields())
    assert np.abs(a - fs["a"]).max() <= 1e-9 * np.abs(fs["phi"]).max() / spec.h[1]
    s.check()
    s.close()


def test_field_step_needs_profiles_and_third_buffer(torch):
    from paper_2212_03036_b200.binding import Sldg, SldgError
    spec = inputs.itg_grid(4, 4, 2, 4, 2)
    s = Sldg(spec)
    with pytest.raises(SldgError):
        s.field_step()
    with pytest.raises(SldgError):
        s._chk(s.L.sldg_step_algorithm2(s.h, 1.0, 1e-12, 10), "sldg_step_algorithm2")
    s.close()

"""Out-of-bounds writes: every device buffer the library gets sits between two margins filled with a byte pattern, every
kernel family runs (all orders, ragged sizes, fused and separate sweeps, streaming and direct 2d apply, field step,
Algorithms 1 and 2, source term, host entry points), and the margins must come back untouched.  (compute-sanitizer is
closed on this pool: "find a bad access with bounds checks and asserts of your own".)"""
import numpy as np
import pytest

from paper_2212_03036_b200 import inputs

pytestmark = pytest.mark.gpu
GUARD = 1 << 20


@pytest.fixture(scope="module")
def torch():
    import torch as t
    if not t.cuda.is_available():
        pytest.skip("needs a CUDA device")
    return t


CASES = [(2, (16, 16, 8, 16)), (3, (9, 7, 3, 8)), (1, (12, 10, 5, 16)), (2, (5, 3, 3, 7)), (3, (4, 5, 2, 5)),
         (2, (40, 36, 2, 72)), (2, (3, 3, 70, 4)), (3, (24, 20, 2, 48))]


@pytest.mark.parametrize("o,cells", CASES)
@pytest.mark.parametrize("fuse", ["plane", "tiled", "separate"])
def test_no_kernel_writes_outside_its_buffers(torch, monkeypatch, o, cells, fuse):
    from paper_2212_03036_b200.binding import Sldg, SldgError
    if fuse == "separate":
        monkeypatch.setenv("SLDG_NO_FUSE", "1")
    if fuse == "tiled":
        monkeypatch.setenv("SLDG_FORCE_TILE", "1")
    spec = inputs.itg_grid(*cells, o)
    f = inputs.itg_initial_f(spec, eps=0.05)
    cu = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
    for layout in (1, 2, 3):
        s = Sldg(spec, layout=layout, guard_bytes=GUARD)
        s.import_state(cu(f))
        a, b, Ez, _ = inputs.itg_fields(spec, 4.0, 0.8)
        s.set_Ez(cu(Ez))
        s.set_vxy(cu(a), cu(b), 1)
        s.advect_z(7.0)           # large Courant numbers: wrap-around paths
        s.advect_v(300.0)
        s.advect_xy(4.0, 1)
        s.advect_xy(4.0, 2)
        s.strang_step(4.0)
        s.charge_density()
        s.mass()
        n0, Te = inputs.itg_vertex_profiles(spec)
        s.set_profiles(cu(n0), cu(Te), 1.0)
        s.field_step(1e-10, 200)
        s.diagnostics(inputs.ITG_RP)
        s.step_algorithm1(0.05, 1e-10, 200)
        s.step_algorithm2(0.05, 1e-10, 200)
        vv = spec.node_coords(3)
        prof = np.repeat((-vv * np.exp(-0.5 * vv * vv))[:, None], spec.N[0], axis=1)
        s.set_equilibrium(cu(prof), cu(-prof))
        s.set_source_fields(cu(Ez), cu(Ez))
        s.strang_step_sources(1.0)
        rho_h = np.empty((spec.N[2], spec.N[1], spec.N[0]))
        mass_h = np.empty(1)
        s.strang_step_host(2.0, Ez, a, b, 1, rho_h, mass_h)
        s.debug_geometry(0)
        s.debug_counter(1)
        s.export_state()
        try:  # a geometry error word (the state went through deliberately wild steps) is not an out-of-bounds write
            s.check()
        except SldgError as e:
            assert e.code in (-3, -4)
        assert s.check_guards(), (o, cells, layout, fuse)
        s.close()


def test_direct_apply_paths_stay_inside(torch, monkeypatch):
    # solid-body rotation sends most blocks to the direct 2d apply; also the forced direct path
    from paper_2212_03036_b200.binding import Sldg
    cu = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
    for o, forced in ((2, False), (3, False), (2, True)):
        if forced:
            monkeypatch.setenv("SLDG_APPLY_DIRECT", "1")
        spec = inputs.bumps_grid(48, 40, o)
        s = Sldg(spec, guard_bytes=GUARD)
        s.import_state(cu(inputs.bumps_initial_f(spec, seed=1)))
        a, b = inputs.rotation_velocity(spec)
        s.set_vxy(cu(a), cu(b), 0)
        for _ in range(3):
            s.advect_xy(0.15, 2)
        s.check()
        assert s.check_guards(), (o, forced)
        s.close()


@pytest.mark.parametrize("o,cells", [(2, (32, 32, 16, 32)), (3, (16, 16, 8, 16)), (2, (24, 20, 3, 72))])
def test_runs_are_bitwise_reproducible(torch, o, cells):
    # races between the producer warp's bulk copies, the in-place sweeps and the ring recycling would show up as
    # run-to-run differences: five fused steps, Algorithm 2 and the source term, three times from the same state
    from paper_2212_03036_b200.binding import Sldg
    spec = inputs.itg_grid(*cells, o)
    f = inputs.itg_initial_f(spec, eps=0.05)
    cu = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
    a, b, Ez, _ = inputs.itg_fields(spec, 4.0, 0.8)
    n0, Te = inputs.itg_vertex_profiles(spec)
    outs = []
    for rep in range(3):
        res = []
        s = Sldg(spec)
        s.import_state(cu(f))
        s.set_Ez(cu(Ez))
        s.set_vxy(cu(a), cu(b), 1)
        for _ in range(5):
            s.strang_step(4.0)
        s.check()
        res.append(s.export_state().cpu().numpy())
        s.close()
        s = Sldg(spec)  # the self-consistent steps start from the smooth initial state (a resolved field)
        s.import_state(cu(f))
        s.set_profiles(cu(n0), cu(Te), 1.0)
        s.step_algorithm2(0.5, 1e-12, 500)
        s.step_algorithm1(0.5, 1e-12, 500)
        s.check()
        res.append(s.export_state().cpu().numpy())
        s.close()
        outs.append(res)
    for k in range(2):
        assert np.array_equal(outs[0][k], outs[1][k]) and np.array_equal(outs[0][k], outs[2][k]), k

"""the swirling-deformation convergence study of the 2d step (Table 1) --
on the CPU oracle (pins the method's order of convergence, a property the paper prints: L2 orders 2.29-2.42 for
k = 1, "error in mass ... close to machine precision") and through the CUDA library (parity of the whole study)."""
import numpy as np
import pytest

import oracle
from paper_2212_03036_b200 import experiments


def _oracle_stepper(spec, f0):
    st = {"f": np.ascontiguousarray(f0).copy()}

    def step(a, b, tau):
        st["f"] = oracle.advect_xy(spec, st["f"], a, b, tau, 2, 1)

    return step, (lambda: st["f"])


@pytest.fixture(scope="module")
def oracle_rows():
    return experiments.swirl_convergence((20, 40, 80), 2, make_stepper=_oracle_stepper)


def test_oracle_swirl_table_has_the_papers_order(oracle_rows):
    # PAPER.md:307-310 prints 5.20e-2, 9.94e-3, 1.85e-3 (orders 2.39, 2.42) for its own cosine bell; the bell's centre
    # and radius are not in the paper, so the errors agree in size and the orders in value, not digit by digit
    for r, paper_l2 in zip(oracle_rows, (5.20e-2, 9.94e-3, 1.85e-3)):
        assert 0.5 * paper_l2 < r["l2"] < 2.0 * paper_l2, r
        assert r["mass_err"] < 1e-13, r
    for r in oracle_rows[1:]:
        assert 2.0 < r["l2_order"] < 2.8, r
        assert 1.7 < r["linf_order"] < 2.8, r


@pytest.mark.gpu
def test_gpu_swirl_table_matches_the_oracle_and_converges(oracle_rows):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    rows = experiments.swirl_convergence((20, 40, 80, 160), 2)
    for g, r in zip(rows, oracle_rows):
        assert g["steps"] == r["steps"]
        assert abs(g["l2"] - r["l2"]) <= 1e-9 * r["l2"], (g, r)
        assert abs(g["linf"] - r["linf"]) <= 1e-9 * r["linf"], (g, r)
    for g in rows:
        assert g["mass_err"] < 1e-13, g
    # the super-convergence of the coarse meshes fades: 160^2 sits at the design order 2 of straight-edged upstream
    # cells traced by the explicit midpoint rule (measured 1.99; the paper, tracing its analytic flow, prints 2.29)
    for g in rows[1:]:
        assert 1.9 < g["l2_order"] < 2.8, g
    rows3 = experiments.swirl_convergence((20, 40, 80), 3)  # o = 3: straight-edged upstream cells cap the order at ~2
    for g in rows3[1:]:
        assert g["l2_order"] > 1.6 and g["mass_err"] < 1e-13, g  # measured on the B200: 1.79 at 80^2

"""CPU-only checks of the C-ABI boundary: libsldg.so builds/loads without a GPU and exports every symbol
include/sldg.h declares; host-only entry points validate parameters.  No compute calls here."""
import ctypes as C
import os
import re

import pytest

from paper_2212_03036_b200 import binding, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "sldg.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sldg_[a-z_A-Z0-9]+)\s*\(", src)))


def test_header_declares_north_star_entry_points():
    names = _declared_functions()
    for must in ("sldg_create", "sldg_advect_z", "sldg_advect_v", "sldg_advect_xy", "sldg_charge_density",
                 "sldg_strang_step"):
        assert must in names


def test_library_exports_every_declared_symbol():
    L = binding.load_library()
    names = _declared_functions()
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), f"libsldg.so does not export {n}"
    assert sorted(binding.EXPORTS) == names


def test_sizes_and_parameter_validation():
    L = binding.load_library()
    spec = inputs.itg_grid(16, 16, 8, 16, 2)
    p = binding.make_params(spec)
    sb = L.sldg_state_bytes(C.byref(p))
    assert sb == spec.dofs * 8  # Nv = 32 needs no padding
    assert L.sldg_workspace_bytes(C.byref(p)) > 0
    # padded v pitch: Nv = 3*7 = 21 -> 32
    spec2 = inputs.GridSpec(n=(4, 4, 2, 7), order=(3, 3, 3, 3), lo=(0, 0, 0, 0), hi=(1, 1, 1, 1))
    p2 = binding.make_params(spec2)
    assert L.sldg_state_bytes(C.byref(p2)) == 12 * 12 * 6 * 32 * 8
    bad = binding.make_params(spec)
    bad.order[0] = 3  # order[0] != order[1]
    assert L.sldg_state_bytes(C.byref(bad)) == 0
    bad = binding.make_params(spec)
    bad.max_stencil = 5
    assert L.sldg_workspace_bytes(C.byref(bad)) == 0
    bad = binding.make_params(spec)
    bad.order[3] = 4
    assert L.sldg_state_bytes(C.byref(bad)) == 0
    h = C.c_void_p()
    assert L.sldg_create(C.byref(p), None, None, None, 0, None, C.byref(h)) == binding.SLDG_EINVAL
    assert L.sldg_strerror(binding.SLDG_ESTENCIL) and L.sldg_strerror(binding.SLDG_EGEOM)


def test_product_path_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError):
        binding.Sldg(inputs.itg_grid(4, 4, 2, 4, 2))

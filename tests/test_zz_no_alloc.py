"""sldg_mass_static, the allocation-free entry point (include/sldg.h, sldg_static.cu): its output against the existing
path (Sldg.import_state + Sldg.mass, caller-allocated workspace) and against the oracle's mass, on two calls in a row
that share the library's static device scratch.  Collected last on purpose (pytest -x): the file
name sorts after every other test file.  Passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from paper_2212_03036_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1e-13  # relative, the mass tolerance of the parity tests


@pytest.fixture(scope="module")
def torch():
    import torch as t
    if not t.cuda.is_available():
        pytest.skip("needs a CUDA device")
    return t


def _existing_path(torch, spec, f_dev):
    from paper_2212_03036_b200.binding import Sldg
    s = Sldg(spec)
    s.import_state(f_dev)
    m = float(s.mass().cpu()[0])
    s.check()
    s.close()
    return m


# the second call of each pair is SMALLER than the first and holds different data: stale scratch of the first call
# (charge density beyond the second grid's nodes, partial sums beyond its block count) must not reach the result
PAIRS = [
    ((2, (16, 16, 8, 16)), (2, (5, 3, 3, 7))),
    ((3, (9, 7, 3, 8)), (1, (12, 10, 5, 16))),
    ((2, (64, 64, 32, 8)), (3, (4, 5, 2, 5))),  # 524288 nodes: 2048 blocks > 1024 partial sums (grid-stride path)
]


@pytest.mark.parametrize("first,second", PAIRS)
def test_two_calls_in_a_row_match_the_existing_path(torch, first, second):
    import oracle
    from paper_2212_03036_b200 import binding
    assert binding.load_library().sldg_mass_static_setup() == 0
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    specs, fs, devs = [], [], []
    for k, (o, cells) in enumerate((first, second)):
        spec = inputs.itg_grid(*cells, o)
        f = inputs.itg_initial_f(spec, eps=0.05 + 0.2 * k)
        specs.append(spec)
        fs.append(f)
        devs.append(torch.from_numpy(np.ascontiguousarray(f)).cuda())
    # two calls back to back on one stream, nothing in between
    binding.mass_static(specs[0], devs[0], out[0:1])
    binding.mass_static(specs[1], devs[1], out[1:2])
    got = out.cpu().numpy()
    for k in range(2):
        want = _existing_path(torch, specs[k], devs[k])
        assert abs(got[k] - want) <= TOL * abs(want), (k, got[k], want)
        if specs[k].dofs <= 1 << 22:
            ref = oracle.mass(specs[k], fs[k])
            assert abs(got[k] - ref) <= TOL * abs(ref), (k, got[k], ref)
    # the same input again: the scratch now holds the second call's leftovers
    again = torch.empty(1, dtype=torch.float64, device="cuda")
    binding.mass_static(specs[0], devs[0], again)
    assert float(again.cpu()[0]) == got[0]  # deterministic: bitwise


def test_calls_leave_device_memory_alone(torch):
    from paper_2212_03036_b200 import binding
    spec = inputs.itg_grid(16, 16, 8, 16, 2)
    f = torch.from_numpy(np.ascontiguousarray(inputs.itg_initial_f(spec))).cuda()
    out = torch.empty(1, dtype=torch.float64, device="cuda")
    binding.mass_static(spec, f, out)  # loads the kernels (lazy module loading may take memory once)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(2):
        binding.mass_static(spec, f, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0


def test_sizes_beyond_the_scratch_are_rejected(torch):
    from paper_2212_03036_b200 import binding
    L = binding.load_library()
    limit = L.sldg_mass_static_max_nodes()
    assert limit == 1 << 20
    # 128 x 128 x 65 nodes = 1,064,960 > 1,048,576; nothing is read before the size check: a tiny buffer stands in
    spec = inputs.GridSpec(n=(64, 64, 65, 1), order=(2, 2, 1, 1), lo=(0, 0, 0, 0), hi=(1, 1, 1, 1))
    p = binding.make_params(spec)
    import ctypes as C
    dummy = torch.zeros(2, dtype=torch.float64, device="cuda")
    rc = L.sldg_mass_static(C.byref(p), dummy.data_ptr(), dummy[1:].data_ptr(), None)
    assert rc == binding.SLDG_ELIMIT
    torch.cuda.synchronize()
    assert float(dummy[1]) == 0.0  # nothing was launched
    # exactly at the limit is accepted
    spec = inputs.GridSpec(n=(64, 64, 64, 1), order=(2, 2, 1, 1), lo=(0, 0, 0, 0), hi=(1, 2, 3, 4))
    f = torch.full(spec.shape, 0.5, dtype=torch.float64, device="cuda")
    out = torch.empty(1, dtype=torch.float64, device="cuda")
    binding.mass_static(spec, f, out)
    assert abs(float(out.cpu()[0]) - 0.5 * 1 * 2 * 3 * 4) <= 1e-12
    # the binding turns the code into a message that names the limit
    big = inputs.GridSpec(n=(64, 64, 65, 1), order=(2, 2, 1, 1), lo=(0, 0, 0, 0), hi=(1, 1, 1, 1))
    with pytest.raises(ValueError, match="exceed the static scratch"):
        fbig = torch.zeros(big.shape, dtype=torch.float64, device="cuda")
        binding.mass_static(big, fbig, out)
    # bad arguments
    assert L.sldg_mass_static(C.byref(p), None, out.data_ptr(), None) == binding.SLDG_EINVAL
    bad = binding.make_params(spec)
    bad.order[3] = 4
    assert L.sldg_mass_static(C.byref(bad), f.data_ptr(), out.data_ptr(), None) == binding.SLDG_EINVAL

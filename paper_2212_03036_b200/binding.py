"""ctypes binding of libsldg (include/sldg.h): same names, argument marshalling only.

Every step of the hot path runs inside the CUDA library.  `Sldg` is a small convenience wrapper that
owns the torch tensors backing the state / workspace and forwards to the C-ABI entry points.
"""
from __future__ import annotations

import ctypes as C
import os

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None

SLDG_OK, SLDG_EINVAL, SLDG_ECUDA, SLDG_ESTENCIL, SLDG_EGEOM = 0, -1, -2, -3, -4
SLDG_ELIMIT = -5

EXPORTS = [
    "sldg_state_bytes", "sldg_workspace_bytes", "sldg_create", "sldg_destroy", "sldg_import_state",
    "sldg_export_state", "sldg_import_state_host", "sldg_export_state_host", "sldg_current",
    "sldg_set_Ez", "sldg_set_vxy", "sldg_advect_z", "sldg_advect_v", "sldg_advect_xy",
    "sldg_charge_density", "sldg_mass", "sldg_strang_step", "sldg_set_trace_order",
    "sldg_strang_step_host", "sldg_check", "sldg_last_timing_ms", "sldg_launch_count",
    "sldg_debug_geometry", "sldg_debug_counter", "sldg_debug_fp64_peak", "sldg_strerror",
    "sldg_set_profiles", "sldg_field_step", "sldg_field_info", "sldg_get_phi", "sldg_get_fields", "sldg_diagnostics",
    "sldg_step_algorithm1", "sldg_set_third_buffer", "sldg_step_algorithm2",
    "sldg_set_equilibrium", "sldg_set_source_fields", "sldg_source_step", "sldg_strang_step_sources",
    "sldg_set_polar_profiles", "sldg_polar_field_step", "sldg_get_polar_phi", "sldg_get_source_fields",
    "sldg_step_algorithm1_polar", "sldg_step_algorithm2_polar", "sldg_timing_history",
    "sldg_mass_static", "sldg_mass_static_setup", "sldg_mass_static_max_nodes",
]


class SldgParams(C.Structure):
    _fields_ = [("n", C.c_int32 * 4), ("order", C.c_int32 * 4), ("lo", C.c_double * 4),
                ("hi", C.c_double * 4), ("max_stencil", C.c_int32), ("layout", C.c_int32)]


class SldgError(RuntimeError):
    def __init__(self, code, what):
        self.code = code
        msg = load_library().sldg_strerror(code).decode()
        super().__init__(f"{what}: {msg} ({code})")


def library_path():
    return os.path.join(_HERE, "libsldg.so")


def load_library():
    """Load libsldg.so (building it with nvcc if the sources are newer).  Raises if unavailable."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    if not os.path.exists(path) or os.environ.get("SLDG_REBUILD"):
        _build.build()
    if not os.path.exists(path):
        raise RuntimeError("libsldg.so is missing and could not be built (nvcc required); "
                           "there is no CPU fallback")
    L = C.CDLL(path)
    vp, dp, ip = C.c_void_p, C.c_void_p, C.c_void_p
    PP = C.POINTER(SldgParams)
    L.sldg_state_bytes.argtypes = [PP]
    L.sldg_state_bytes.restype = C.c_size_t
    L.sldg_workspace_bytes.argtypes = [PP]
    L.sldg_workspace_bytes.restype = C.c_size_t
    L.sldg_create.argtypes = [PP, dp, dp, vp, C.c_size_t, vp, C.POINTER(vp)]
    L.sldg_destroy.argtypes = [vp]
    for name in ("sldg_import_state", "sldg_export_state", "sldg_import_state_host",
                 "sldg_export_state_host", "sldg_set_Ez", "sldg_charge_density", "sldg_mass"):
        getattr(L, name).argtypes = [vp, dp]
    L.sldg_current.argtypes = [vp]
    L.sldg_current.restype = C.c_void_p
    L.sldg_set_vxy.argtypes = [vp, dp, dp, C.c_int]
    L.sldg_advect_z.argtypes = [vp, C.c_double]
    L.sldg_advect_v.argtypes = [vp, C.c_double]
    L.sldg_advect_xy.argtypes = [vp, C.c_double, C.c_int]
    L.sldg_strang_step.argtypes = [vp, C.c_double]
    L.sldg_set_trace_order.argtypes = [vp, C.c_int]
    L.sldg_strang_step_host.argtypes = [vp, C.c_double, dp, dp, dp, C.c_int, dp, dp]
    L.sldg_check.argtypes = [vp]
    L.sldg_last_timing_ms.argtypes = [vp, C.POINTER(C.c_float * 8)]
    L.sldg_launch_count.argtypes = [vp]
    L.sldg_timing_history.argtypes = [vp, C.c_int, C.POINTER(C.c_float)]
    L.sldg_launch_count.restype = C.c_longlong
    L.sldg_debug_geometry.argtypes = [vp, C.c_int, ip, ip, dp]
    L.sldg_debug_counter.argtypes = [vp, C.c_int, C.POINTER(C.c_longlong)]
    L.sldg_debug_fp64_peak.argtypes = [vp, C.c_int, C.POINTER(C.c_double)]
    L.sldg_strerror.argtypes = [C.c_int]
    L.sldg_strerror.restype = C.c_char_p
    L.sldg_set_profiles.argtypes = [vp, dp, dp, C.c_double]
    L.sldg_field_step.argtypes = [vp, C.c_double, C.c_int]
    L.sldg_field_info.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_double)]
    L.sldg_get_phi.argtypes = [vp, dp]
    L.sldg_get_fields.argtypes = [vp, dp, dp, dp]
    L.sldg_diagnostics.argtypes = [vp, C.c_double, C.POINTER(C.c_double * 5)]
    L.sldg_step_algorithm1.argtypes = [vp, C.c_double, C.c_double, C.c_int]
    L.sldg_set_third_buffer.argtypes = [vp, dp]
    L.sldg_step_algorithm2.argtypes = [vp, C.c_double, C.c_double, C.c_int]
    L.sldg_set_equilibrium.argtypes = [vp, dp, dp]
    L.sldg_set_source_fields.argtypes = [vp, dp, dp]
    L.sldg_source_step.argtypes = [vp, C.c_double]
    L.sldg_strang_step_sources.argtypes = [vp, C.c_double]
    L.sldg_set_polar_profiles.argtypes = [vp, dp, dp, dp]
    L.sldg_polar_field_step.argtypes = [vp]
    L.sldg_get_polar_phi.argtypes = [vp, dp]
    L.sldg_get_source_fields.argtypes = [vp, dp, dp]
    L.sldg_step_algorithm1_polar.argtypes = [vp, C.c_double]
    L.sldg_step_algorithm2_polar.argtypes = [vp, C.c_double]
    L.sldg_mass_static.argtypes = [PP, dp, dp, vp]
    L.sldg_mass_static_setup.argtypes = []
    L.sldg_mass_static_max_nodes.argtypes = []
    L.sldg_mass_static_max_nodes.restype = C.c_longlong
    _lib = L
    return L


def make_params(spec, layout=0, max_stencil=3):
    p = SldgParams()
    for d in range(4):
        p.n[d] = int(spec.n[d])
        p.order[d] = int(spec.order[d])
        p.lo[d] = float(spec.lo[d])
        p.hi[d] = float(spec.hi[d])
    p.max_stencil = max_stencil
    p.layout = layout
    return p


def mass_static(spec, f_canonical, out, stream=None):
    """sldg_mass_static: total mass of a canonical-layout distribution into the one-element CUDA tensor `out`, with no
    context, no workspace and no allocation (the scratch is a static device array inside libsldg.so).  Calls on one
    stream are ordered; calls that overlap on the GPU race on the shared scratch."""
    import torch

    if not torch.cuda.is_available():
        raise RuntimeError("libsldg needs a CUDA device (sm_100a); there is no CPU fallback")
    L = load_library()
    assert f_canonical.is_cuda and f_canonical.dtype == torch.float64 and f_canonical.is_contiguous()
    assert tuple(f_canonical.shape) == tuple(spec.shape)
    assert out.is_cuda and out.dtype == torch.float64 and out.numel() == 1 and out.device == f_canonical.device
    p = make_params(spec)
    with torch.cuda.device(f_canonical.device):
        st = stream if stream is not None else torch.cuda.current_stream()
        rc = L.sldg_mass_static(C.byref(p), f_canonical.data_ptr(), out.data_ptr(), st.cuda_stream)
    if rc == SLDG_ELIMIT:
        N = [int(spec.n[d]) * int(spec.order[d]) for d in range(3)]
        raise ValueError(f"sldg_mass_static: Nx*Ny*Nz = {N[0] * N[1] * N[2]} nodes exceed the static scratch of "
                         f"{L.sldg_mass_static_max_nodes()} nodes; use Sldg.mass() (caller-allocated workspace)")
    if rc != 0:
        raise SldgError(rc, "sldg_mass_static")
    return out


class Sldg:
    """One SLDG context on the current CUDA device.  Tensors are torch CUDA tensors (fp64)."""

    def __init__(self, spec, device="cuda", layout=0, stream=None, guard_bytes=0):
        """guard_bytes > 0 (a multiple of 256): every device buffer handed to the library is the middle of a larger
        allocation whose margins are filled with a byte pattern; check_guards() verifies that no kernel wrote outside
        its buffers (the pool's compute-sanitizer is closed: DESIGN.md section 12)."""
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("libsldg needs a CUDA device (sm_100a); there is no CPU fallback")
        self.torch = torch
        self.L = load_library()
        self.spec = spec
        self.device = torch.device(device)
        self.params = make_params(spec, layout)
        sb = self.L.sldg_state_bytes(C.byref(self.params))
        wb = self.L.sldg_workspace_bytes(C.byref(self.params))
        if sb == 0 or wb == 0:
            raise SldgError(SLDG_EINVAL, "sldg_state_bytes")
        self.state_bytes, self.workspace_bytes = sb, wb
        assert guard_bytes % 256 == 0
        self.guard_bytes = guard_bytes
        self._guarded = []

        def alloc(nbytes):
            if guard_bytes == 0:
                return torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            raw = torch.full((nbytes + 2 * guard_bytes,), 0xA5, dtype=torch.uint8, device=self.device)
            self._guarded.append(raw)
            return raw[guard_bytes:guard_bytes + nbytes]

        self.f_a = alloc(sb).view(torch.float64)
        self.f_b = alloc(sb).view(torch.float64)
        self.workspace = alloc(wb)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            rc = self.L.sldg_create(C.byref(self.params), self.f_a.data_ptr(), self.f_b.data_ptr(),
                                    self.workspace.data_ptr(), wb, self.stream.cuda_stream, C.byref(h))
        self._chk(rc, "sldg_create")
        self.h = h

    def _chk(self, rc, what):
        if rc != 0:
            raise SldgError(rc, what)

    def check_guards(self):
        """True if the margins around every buffer still hold their pattern (always True without guard_bytes)."""
        self.torch.cuda.synchronize(self.device)
        g = self.guard_bytes
        return all(bool((raw[:g] == 0xA5).all()) and bool((raw[raw.numel() - g:] == 0xA5).all()) for raw in self._guarded) if g else True

    def close(self):
        if getattr(self, "h", None):
            self.L.sldg_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- state ---------------------------------------------------------------------------------
    def import_state(self, f_canonical):
        assert f_canonical.is_cuda and f_canonical.dtype == self.torch.float64 and f_canonical.is_contiguous()
        assert tuple(f_canonical.shape) == tuple(self.spec.shape)
        self._chk(self.L.sldg_import_state(self.h, f_canonical.data_ptr()), "sldg_import_state")

    def export_state(self, out=None):
        if out is None:
            out = self.torch.empty(self.spec.shape, dtype=self.torch.float64, device=self.device)
        self._chk(self.L.sldg_export_state(self.h, out.data_ptr()), "sldg_export_state")
        return out

    def import_state_host(self, f_host):
        """f_host: numpy array or CPU torch tensor, canonical layout."""
        ptr = f_host.ctypes.data if hasattr(f_host, "ctypes") else f_host.data_ptr()
        self._chk(self.L.sldg_import_state_host(self.h, ptr), "sldg_import_state_host")

    def export_state_host(self, f_host):
        ptr = f_host.ctypes.data if hasattr(f_host, "ctypes") else f_host.data_ptr()
        self._chk(self.L.sldg_export_state_host(self.h, ptr), "sldg_export_state_host")
        return f_host

    def current_ptr(self):
        return self.L.sldg_current(self.h)

    # ---- fields --------------------------------------------------------------------------------
    def set_Ez(self, Ez):
        assert Ez.is_cuda and Ez.dtype == self.torch.float64 and Ez.is_contiguous()
        self._chk(self.L.sldg_set_Ez(self.h, Ez.data_ptr()), "sldg_set_Ez")

    def set_vxy(self, a, b, periodic):
        for u in (a, b):
            assert u.is_cuda and u.dtype == self.torch.float64 and u.is_contiguous()
        self._chk(self.L.sldg_set_vxy(self.h, a.data_ptr(), b.data_ptr(), int(periodic)), "sldg_set_vxy")

    def set_trace_order(self, order):
        self._chk(self.L.sldg_set_trace_order(self.h, int(order)), "sldg_set_trace_order")

    # ---- substeps ------------------------------------------------------------------------------
    def advect_z(self, tau):
        self._chk(self.L.sldg_advect_z(self.h, float(tau)), "sldg_advect_z")

    def advect_v(self, tau):
        self._chk(self.L.sldg_advect_v(self.h, float(tau)), "sldg_advect_v")

    def advect_xy(self, tau, trace_order=2):
        self._chk(self.L.sldg_advect_xy(self.h, float(tau), int(trace_order)), "sldg_advect_xy")

    def strang_step(self, dt):
        self._chk(self.L.sldg_strang_step(self.h, float(dt)), "sldg_strang_step")

    def strang_step_host(self, dt, Ez_host=None, a_host=None, b_host=None, periodic=1, rho_host=None,
                         mass_host=None):
        def ptr(x):
            if x is None:
                return None
            return x.ctypes.data if hasattr(x, "ctypes") else x.data_ptr()
        self._chk(self.L.sldg_strang_step_host(self.h, float(dt), ptr(Ez_host), ptr(a_host), ptr(b_host),
                                               int(periodic), ptr(rho_host), ptr(mass_host)),
                  "sldg_strang_step_host")

    def charge_density(self, out=None):
        Nz, Nv, Ny, Nx = self.spec.shape
        if out is None:
            out = self.torch.empty((Nz, Ny, Nx), dtype=self.torch.float64, device=self.device)
        self._chk(self.L.sldg_charge_density(self.h, out.data_ptr()), "sldg_charge_density")
        return out

    def mass(self, out=None):
        if out is None:
            out = self.torch.empty(1, dtype=self.torch.float64, device=self.device)
        self._chk(self.L.sldg_mass(self.h, out.data_ptr()), "sldg_mass")
        return out

    # ---- field step, invariants, Algorithms 1 and 2 -------------------------------------------------
    def set_profiles(self, n0, Te, B=1.0):
        for u in (n0, Te):
            assert u.is_cuda and u.dtype == self.torch.float64 and u.is_contiguous()
        self._chk(self.L.sldg_set_profiles(self.h, n0.data_ptr(), Te.data_ptr(), float(B)), "sldg_set_profiles")

    def field_step(self, tol=1e-13, max_iter=2000):
        self._chk(self.L.sldg_field_step(self.h, float(tol), int(max_iter)), "sldg_field_step")

    def field_info(self):
        it, rr = C.c_int(0), C.c_double(0.0)
        self._chk(self.L.sldg_field_info(self.h, C.byref(it), C.byref(rr)), "sldg_field_info")
        return int(it.value), float(rr.value)

    def get_phi(self):
        nx, ny = self.spec.n[0], self.spec.n[1]
        out = self.torch.empty((self.spec.N[2], ny, nx), dtype=self.torch.float64, device=self.device)
        self._chk(self.L.sldg_get_phi(self.h, out.data_ptr()), "sldg_get_phi")
        return out

    def get_fields(self):
        t = self.torch
        Nx, Ny, Nz, _ = self.spec.N
        nx, ny = self.spec.n[0], self.spec.n[1]
        Ez = t.empty((Nz, Ny, Nx), dtype=t.float64, device=self.device)
        a = t.empty((Nz, ny + 1, nx + 1), dtype=t.float64, device=self.device)
        b = t.empty_like(a)
        self._chk(self.L.sldg_get_fields(self.h, Ez.data_ptr(), a.data_ptr(), b.data_ptr()), "sldg_get_fields")
        return Ez, a, b

    def diagnostics(self, r_p):
        out = (C.c_double * 5)()
        self._chk(self.L.sldg_diagnostics(self.h, float(r_p), C.byref(out)), "sldg_diagnostics")
        return dict(zip(("electric", "mass", "l2", "kinetic", "potential"), (float(x) for x in out)))

    def step_algorithm1(self, dt, tol=1e-13, max_iter=2000):
        self._chk(self.L.sldg_step_algorithm1(self.h, float(dt), float(tol), int(max_iter)), "sldg_step_algorithm1")

    def step_algorithm2_polar(self, dt):
        self._third_buffer()
        self._chk(self.L.sldg_step_algorithm2_polar(self.h, float(dt)), "sldg_step_algorithm2_polar")

    def step_algorithm2(self, dt, tol=1e-13, max_iter=2000):
        self._third_buffer()
        self._chk(self.L.sldg_step_algorithm2(self.h, float(dt), float(tol), int(max_iter)), "sldg_step_algorithm2")

    def _third_buffer(self):
        if getattr(self, "f_c", None) is None:  # the third copy of f
            g = self.guard_bytes
            if g == 0:
                self.f_c = self.torch.empty(self.state_bytes // 8, dtype=self.torch.float64, device=self.device)
            else:
                raw = self.torch.full((self.state_bytes + 2 * g,), 0xA5, dtype=self.torch.uint8, device=self.device)
                self._guarded.append(raw)
                self.f_c = raw[g:g + self.state_bytes].view(self.torch.float64)
            self._chk(self.L.sldg_set_third_buffer(self.h, self.f_c.data_ptr()), "sldg_set_third_buffer")

    # ---- delta-g formulation: source term (polar coordinates, axis 0 = r, axis 1 = theta) ------------
    def set_equilibrium(self, dv_geq, dr_geq):
        for u in (dv_geq, dr_geq):
            assert u.is_cuda and u.dtype == self.torch.float64 and u.is_contiguous()
        self._chk(self.L.sldg_set_equilibrium(self.h, dv_geq.data_ptr(), dr_geq.data_ptr()), "sldg_set_equilibrium")

    def set_source_fields(self, dz_phi, dtheta_phi):
        for u in (dz_phi, dtheta_phi):
            assert u.is_cuda and u.dtype == self.torch.float64 and u.is_contiguous()
        self._chk(self.L.sldg_set_source_fields(self.h, dz_phi.data_ptr(), dtheta_phi.data_ptr()), "sldg_set_source_fields")

    def source_step(self, tau):
        self._chk(self.L.sldg_source_step(self.h, float(tau)), "sldg_source_step")

    def strang_step_sources(self, dt):
        self._chk(self.L.sldg_strang_step_sources(self.h, float(dt)), "sldg_strang_step_sources")

    def set_polar_profiles(self, r_n0, dln_n0, Te):
        for u in (r_n0, dln_n0, Te):
            assert u.is_cuda and u.dtype == self.torch.float64 and u.is_contiguous() and u.numel() == self.spec.n[0] + 1
        self._chk(self.L.sldg_set_polar_profiles(self.h, r_n0.data_ptr(), dln_n0.data_ptr(), Te.data_ptr()), "sldg_set_polar_profiles")

    def polar_field_step(self):
        self._chk(self.L.sldg_polar_field_step(self.h), "sldg_polar_field_step")

    def get_polar_phi(self):
        out = self.torch.empty((self.spec.N[2], self.spec.n[1], self.spec.n[0] + 1), dtype=self.torch.float64, device=self.device)
        self._chk(self.L.sldg_get_polar_phi(self.h, out.data_ptr()), "sldg_get_polar_phi")
        return out

    def get_source_fields(self):
        t = self.torch
        Nx, Ny, Nz, _ = self.spec.N
        dz = t.empty((Nz, Ny, Nx), dtype=t.float64, device=self.device)
        dth = t.empty_like(dz)
        self._chk(self.L.sldg_get_source_fields(self.h, dz.data_ptr(), dth.data_ptr()), "sldg_get_source_fields")
        return dz, dth

    def step_algorithm1_polar(self, dt):
        self._chk(self.L.sldg_step_algorithm1_polar(self.h, float(dt)), "sldg_step_algorithm1_polar")

    # ---- diagnostics ---------------------------------------------------------------------------
    def check(self):
        """Synchronise and raise on a sticky device error."""
        self._chk(self.L.sldg_check(self.h), "sldg_check")

    def last_timing_ms(self):
        ms = (C.c_float * 8)()
        self._chk(self.L.sldg_last_timing_ms(self.h, C.byref(ms)), "sldg_last_timing_ms")
        return list(ms)

    def timing_history(self, n):
        """Per-kernel device times of the last n Strang steps, n x 8 (see sldg_last_timing_ms), oldest first."""
        buf = (C.c_float * (8 * n))()
        self._chk(self.L.sldg_timing_history(self.h, int(n), buf), "sldg_timing_history")
        return [list(buf[8 * i:8 * i + 8]) for i in range(n)]

    def launch_count(self):
        return int(self.L.sldg_launch_count(self.h))

    def debug_counter(self, which=0):
        v = C.c_longlong(0)
        self._chk(self.L.sldg_debug_counter(self.h, int(which), C.byref(v)), "sldg_debug_counter")
        return int(v.value)

    def debug_fp64_peak(self, repeats=5):
        """Measured fp64 FMA throughput of the device in TFLOP/s (the roof of the ALU-bound kernels)."""
        v = C.c_double(0.0)
        self._chk(self.L.sldg_debug_fp64_peak(self.h, int(repeats), C.byref(v)), "sldg_debug_fp64_peak")
        return float(v.value)

    def debug_geometry(self, z):
        t = self.torch
        nx, ny = self.spec.n[0], self.spec.n[1]
        o4 = self.spec.order[0] ** 4
        anchor = t.empty((ny * nx, 2), dtype=t.int32, device=self.device)
        mask = t.empty(ny * nx, dtype=t.int32, device=self.device)
        W = t.empty((ny * nx, 9, o4), dtype=t.float64, device=self.device)
        self._chk(self.L.sldg_debug_geometry(self.h, int(z), anchor.data_ptr(), mask.data_ptr(), W.data_ptr()),
                  "sldg_debug_geometry")
        return anchor, mask, W

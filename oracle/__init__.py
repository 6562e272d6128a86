"""CPU oracle for the SLDG hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes wrapper over oracle/sldg_oracle.c (plain C, fp64, written from the paper; see that file's
header).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2212_03036_b200 except, in callers, the seeded
input generators (paper_2212_03036_b200.inputs holds no arithmetic of the method).

Parity pins: every function is pinned in tests/test_oracle_1d.py and tests/test_oracle_2d.py (list in
DESIGN.md, "Oracle pins").  The rows beyond the hot path have their own modules, same rules: oracle/field.py (Cartesian
field step, invariants, Algorithms 1 and 2; pins in tests/test_oracle_field.py) and oracle/polar.py (source term, the
paper's polar quasi-neutrality solver, the delta-g algorithms; pins in tests/test_oracle_polar.py).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None


class _Grid(C.Structure):
    _fields_ = [("n", C.c_int32 * 4), ("order", C.c_int32 * 4), ("lo", C.c_double * 4),
                ("hi", C.c_double * 4)]


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        P = C.POINTER(C.c_double)
        G = C.POINTER(_Grid)
        L.sldg_oracle_gl.argtypes = [C.c_int, P, P]
        L.sldg_oracle_gl.restype = None
        L.sldg_oracle_shift_matrices.argtypes = [C.c_int, C.c_double, P, P]
        L.sldg_oracle_shift_matrices.restype = None
        L.sldg_oracle_shift_line.argtypes = [C.c_int, C.c_int, C.c_double, P, P]
        L.sldg_oracle_shift_line.restype = None
        L.sldg_oracle_advect_z.argtypes = [G, P, P, C.c_double]
        L.sldg_oracle_advect_v.argtypes = [G, P, P, P, C.c_double]
        L.sldg_oracle_charge_density.argtypes = [G, P, P]
        L.sldg_oracle_mass.argtypes = [G, P]
        L.sldg_oracle_mass.restype = C.c_double
        L.sldg_oracle_cell_coefficients.argtypes = [C.c_int, P, P, C.c_int, C.c_int, P]
        L.sldg_oracle_xy_plane_geometry.argtypes = [G, P, P, C.c_double, C.c_int, C.c_int,
                                                    C.POINTER(C.c_long), C.POINTER(C.c_int32),
                                                    C.POINTER(C.c_int32), P]
        L.sldg_oracle_xy_plane_geometry.restype = C.c_long
        L.sldg_oracle_advect_xy.argtypes = [G, P, P, P, P, C.c_double, C.c_int, C.c_int]
        L.sldg_oracle_strang_step.argtypes = [G, P, P, P, P, P, C.c_double, C.c_int, C.c_int]
        L.sldg_oracle_num_threads.restype = C.c_int
        L.sldg_oracle_trace.argtypes = [G, P, P, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                        C.c_int, C.c_int, P]
        L.sldg_oracle_trace.restype = None
        _lib = L
    return _lib


def _grid(spec):
    g = _Grid()
    for d in range(4):
        g.n[d] = int(spec.n[d])
        g.order[d] = int(spec.order[d])
        g.lo[d] = float(spec.lo[d])
        g.hi[d] = float(spec.hi[d])
    return g


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


class OracleError(RuntimeError):
    pass


def _check(rc, what):
    if rc < 0:
        raise OracleError(f"{what}: oracle error {rc}")


def num_threads():
    return int(lib().sldg_oracle_num_threads())


def gl(n):
    """Gauss-Legendre nodes on (0,1) and weights summing to 1."""
    x = np.empty(n)
    w = np.empty(n)
    lib().sldg_oracle_gl(n, _dp(x), _dp(w))
    return x, w


def shift_matrices(o, alpha):
    """A(alpha), B(alpha) of eq. (11), o x o row-major."""
    A = np.empty((o, o))
    B = np.empty((o, o))
    lib().sldg_oracle_shift_matrices(o, float(alpha), _dp(A), _dp(B))
    return A, B


def shift_line(u, o, delta):
    """One periodic line of len(u)/o cells shifted by the Courant number delta = a*tau/h."""
    u = _c(u)
    out = np.empty_like(u)
    lib().sldg_oracle_shift_line(u.size // o, o, float(delta), _dp(u), _dp(out))
    return out


def advect_z(spec, f, tau):
    f = _c(f)
    assert f.shape == spec.shape
    out = np.empty_like(f)
    _check(lib().sldg_oracle_advect_z(_grid(spec), _dp(f), _dp(out), float(tau)), "advect_z")
    return out


def advect_v(spec, f, Ez, tau):
    f = _c(f)
    Ez = _c(Ez)
    assert f.shape == spec.shape
    out = np.empty_like(f)
    _check(lib().sldg_oracle_advect_v(_grid(spec), _dp(f), _dp(Ez), _dp(out), float(tau)), "advect_v")
    return out


def charge_density(spec, f):
    f = _c(f)
    Nz, Nv, Ny, Nx = spec.shape
    rho = np.empty((Nz, Ny, Nx))
    _check(lib().sldg_oracle_charge_density(_grid(spec), _dp(f), _dp(rho)), "charge_density")
    return rho


def mass(spec, f):
    f = _c(f)
    return float(lib().sldg_oracle_mass(_grid(spec), _dp(f)))


def cell_coefficients(o, corner_feet, node_feet, r, s):
    """C[m][k] of eq. (18) for one target cell and the source cell at offset (r,s); cell units."""
    cf = _c(corner_feet).reshape(4, 2)
    nf = _c(node_feet).reshape(o * o, 2)
    out = np.empty((o * o, o * o))
    rc = lib().sldg_oracle_cell_coefficients(o, _dp(cf), _dp(nf), int(r), int(s), _dp(out))
    _check(rc, "cell_coefficients")
    return out, rc


def trace(spec, a_plane, b_plane, i, j, xi, eta, tau, trace_order=2, vel_periodic=0):
    """Foot of the characteristic through local (xi,eta) of cell (i,j), relative to that cell, cell units."""
    a = _c(a_plane)
    b = _c(b_plane)
    out = np.empty(2)
    lib().sldg_oracle_trace(_grid(spec), _dp(a), _dp(b), int(i), int(j), float(xi), float(eta), float(tau),
                            int(trace_order), int(vel_periodic), _dp(out))
    return out


def xy_plane_geometry(spec, a_plane, b_plane, tau, trace_order=2, vel_periodic=0):
    """Geometry of one z-plane.  Returns (offs[ncell+1], r[ne], s[ne], C[ne][o2][o2])."""
    a = _c(a_plane)
    b = _c(b_plane)
    nx, ny = spec.n[0], spec.n[1]
    assert a.shape == (ny + 1, nx + 1) and b.shape == a.shape
    o2 = spec.order[0] ** 2
    g = _grid(spec)
    ne = lib().sldg_oracle_xy_plane_geometry(g, _dp(a), _dp(b), float(tau), int(trace_order),
                                             int(vel_periodic), None, None, None, None)
    _check(ne, "xy_plane_geometry")
    offs = np.empty(nx * ny + 1, dtype=np.int64)
    er = np.empty(ne, dtype=np.int32)
    es = np.empty(ne, dtype=np.int32)
    eC = np.empty((ne, o2, o2))
    rc = lib().sldg_oracle_xy_plane_geometry(
        g, _dp(a), _dp(b), float(tau), int(trace_order), int(vel_periodic),
        offs.ctypes.data_as(C.POINTER(C.c_long)), er.ctypes.data_as(C.POINTER(C.c_int32)),
        es.ctypes.data_as(C.POINTER(C.c_int32)), _dp(eC))
    _check(rc, "xy_plane_geometry")
    return offs, er, es, eC


def advect_xy(spec, f, a, b, tau, trace_order=2, vel_periodic=0):
    f = _c(f)
    a = _c(a)
    b = _c(b)
    assert f.shape == spec.shape
    Nz = spec.shape[0]
    assert a.shape == (Nz, spec.n[1] + 1, spec.n[0] + 1) and b.shape == a.shape
    out = np.empty_like(f)
    _check(lib().sldg_oracle_advect_xy(_grid(spec), _dp(f), _dp(a), _dp(b), _dp(out), float(tau),
                                       int(trace_order), int(vel_periodic)), "advect_xy")
    return out


def strang_step(spec, f, Ez, a, b, dt, trace_order=2, vel_periodic=0, tmp=None):
    """One Strang step z(dt/2) v(dt/2) xy(dt) v(dt/2) z(dt/2); f is updated IN PLACE and returned."""
    assert f.dtype == np.float64 and f.flags.c_contiguous and f.shape == spec.shape
    Ez = _c(Ez)
    a = _c(a)
    b = _c(b)
    if tmp is None:
        tmp = np.empty_like(f)
    _check(lib().sldg_oracle_strang_step(_grid(spec), _dp(f), _dp(tmp), _dp(Ez), _dp(a), _dp(b),
                                         float(dt), int(trace_order), int(vel_periodic)), "strang_step")
    return f

"""ctypes wrapper around oracle/streams_oracle.cpp -- TEST INFRASTRUCTURE ONLY.

Argument marshalling only; every number comes from the C++ oracle.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_c_double_p = C.POINTER(C.c_double)
_c_ubyte_p = C.POINTER(C.c_ubyte)

DBG_WENO_LINEAR = 1
DBG_NO_PRESSURE = 2
PART_X, PART_Y, PART_Z, PART_VISC, PART_FORCE, PART_ALL = 1, 2, 4, 8, 16, 31


class OracleParams(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
        ("bc_x", C.c_int), ("bc_y_lo", C.c_int), ("bc_y_hi", C.c_int), ("bc_z", C.c_int),
        ("visc_law", C.c_int),
        ("central_order", C.c_int), ("weno_order", C.c_int), ("visc_order", C.c_int), ("flux_mode", C.c_int),
        ("dt_every", C.c_int),
        ("dbg_flags", C.c_int),
        ("lx", C.c_double), ("ly", C.c_double), ("lz", C.c_double),
        ("y_lo", C.c_double), ("y_hi", C.c_double),
        ("t_wall_lo", C.c_double), ("t_wall_hi", C.c_double),
        ("gamma", C.c_double), ("rgas", C.c_double), ("prandtl", C.c_double),
        ("mu_ref", C.c_double), ("t_ref", C.c_double), ("suth_s", C.c_double), ("pow_exp", C.c_double),
        ("u_ref", C.c_double), ("l_ref", C.c_double),
        ("freestream", C.c_double * 5),
        ("sensor_threshold", C.c_double), ("weno_eps", C.c_double),
        ("cfl", C.c_double), ("dt_fixed", C.c_double),
        ("accel", C.c_double * 3),
        ("weno_variant", C.c_int),
    ]


_libs = {}


def load(kind: str = "omp"):
    if kind not in _libs:
        _build.build()
        lib = C.CDLL(_build.lib_path(kind))
        lib.oracle_create.restype = C.c_void_p
        lib.oracle_create.argtypes = [C.POINTER(OracleParams), _c_double_p]
        lib.oracle_destroy.argtypes = [C.c_void_p]
        lib.oracle_ng.argtypes = [C.c_void_p]
        lib.oracle_set_fields.argtypes = [C.c_void_p, _c_double_p]
        lib.oracle_get_fields.argtypes = [C.c_void_p, _c_double_p]
        lib.oracle_rhs.argtypes = [C.c_void_p, C.c_int, _c_double_p]
        lib.oracle_step.argtypes = [C.c_void_p, C.c_int, _c_double_p, _c_double_p]
        lib.oracle_step_forced.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, _c_double_p, _c_double_p, _c_double_p]
        lib.oracle_bulk_sums.argtypes = [C.c_void_p, C.c_int, _c_double_p, _c_double_p]
        lib.oracle_compute_dt.restype = C.c_double
        lib.oracle_compute_dt.argtypes = [C.c_void_p]
        lib.oracle_get_sensor.argtypes = [C.c_void_p, _c_double_p, _c_ubyte_p, _c_double_p]
        lib.oracle_set_mask_override.argtypes = [C.c_void_p, _c_ubyte_p]
        lib.oracle_interface_flags.argtypes = [C.c_void_p, C.c_int, _c_ubyte_p]
        lib.oracle_get_prim.argtypes = [C.c_void_p, C.c_int, _c_double_p]
        lib.oracle_get_padded.argtypes = [C.c_void_p, C.c_int, _c_double_p]
        lib.oracle_get_metrics.argtypes = [C.c_void_p, _c_double_p, _c_double_p, _c_double_p, _c_double_p]
        lib.oracle_fd_coeffs.argtypes = [C.c_int, _c_double_p, _c_double_p]
        lib.oracle_weno_reconstruct.restype = C.c_double
        lib.oracle_weno_reconstruct.argtypes = [_c_double_p, C.c_int, C.c_double, C.c_int, _c_double_p]
        lib.oracle_weno_reconstruct_variant.restype = C.c_double
        lib.oracle_weno_reconstruct_variant.argtypes = [_c_double_p, C.c_int, C.c_double, C.c_int]
        lib.oracle_eigenvectors.argtypes = [C.c_int, _c_double_p, C.c_double, C.c_double, _c_double_p, _c_double_p]
        lib.oracle_num_threads.restype = C.c_int
        _libs[kind] = lib
    return _libs[kind]


def _dp(a):
    return a.ctypes.data_as(_c_double_p)


def params_from_case(case, dbg_flags: int = 0) -> OracleParams:
    p = OracleParams()
    for name in ("nx", "ny", "nz", "bc_x", "bc_y_lo", "bc_y_hi", "bc_z", "visc_law", "central_order",
                 "weno_order", "visc_order", "flux_mode", "dt_every", "lx", "ly", "lz", "t_wall_lo",
                 "t_wall_hi", "gamma", "rgas", "prandtl", "mu_ref", "t_ref", "pow_exp", "u_ref", "l_ref",
                 "sensor_threshold", "weno_eps", "cfl", "dt_fixed"):
        setattr(p, name, getattr(case, name))
    p.y_lo, p.y_hi = case.y_wall_lo, case.y_wall_hi
    p.suth_s = case.suth_s_over_tref
    p.dbg_flags = dbg_flags
    for q in range(5):
        p.freestream[q] = case.freestream[q]
    for a in range(3):
        p.accel[a] = case.accel[a]
    p.weno_variant = case.weno_variant
    return p


class Oracle:
    """One oracle solver instance for a workloads.Case."""

    def __init__(self, case, kind: str = "omp", dbg_flags: int = 0):
        self.lib = load(kind)
        self.case = case
        self.shape = (case.nz, case.ny, case.nx)
        self._y = None if case.y_nodes is None else np.ascontiguousarray(case.y_nodes, dtype=np.float64)
        p = params_from_case(case, dbg_flags)
        self.h = self.lib.oracle_create(C.byref(p), None if self._y is None else _dp(self._y))
        if not self.h:
            raise ValueError("oracle_create rejected the parameters")
        self.ng = self.lib.oracle_ng(self.h)
        if case.w0 is not None:
            self.set_fields(case.w0)

    def close(self):
        if self.h:
            self.lib.oracle_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_fields(self, w):
        w = np.ascontiguousarray(w, dtype=np.float64)
        assert w.shape == (5,) + self.shape
        self.lib.oracle_set_fields(self.h, _dp(w))

    def get_fields(self):
        out = np.empty((5,) + self.shape)
        self.lib.oracle_get_fields(self.h, _dp(out))
        return out

    def rhs(self, parts: int = PART_ALL):
        out = np.empty((5,) + self.shape)
        rc = self.lib.oracle_rhs(self.h, parts, _dp(out))
        if rc:
            raise RuntimeError(f"oracle_rhs rc={rc}")
        return out

    def step(self, nsteps: int):
        dt, t = C.c_double(), C.c_double()
        rc = self.lib.oracle_step(self.h, nsteps, C.byref(dt), C.byref(t))
        if rc:
            raise RuntimeError(f"oracle_step rc={rc}")
        return dt.value, t.value

    def step_forced(self, nsteps: int, direction: int = 0, target: float = float("nan")):
        """nsteps steps under the bulk-flow controller (S18); returns (dt, time, [g_x, g_y, g_z])."""
        dt, t = C.c_double(), C.c_double()
        g = (C.c_double * 3)()
        rc = self.lib.oracle_step_forced(self.h, nsteps, direction, C.c_double(target), C.byref(dt), C.byref(t),
                                         C.cast(g, _c_double_p))
        if rc:
            raise RuntimeError(f"oracle_step_forced rc={rc}")
        return dt.value, t.value, list(g)

    def bulk_sums(self, direction: int = 0):
        m, p = C.c_double(), C.c_double()
        self.lib.oracle_bulk_sums(self.h, direction, C.byref(m), C.byref(p))
        return m.value, p.value

    def compute_dt(self):
        return self.lib.oracle_compute_dt(self.h)

    def sensor(self):
        th = np.empty(self.shape)
        mk = np.empty(self.shape, dtype=np.uint8)
        dv = np.empty(self.shape)
        self.lib.oracle_get_sensor(self.h, _dp(th), mk.ctypes.data_as(_c_ubyte_p), _dp(dv))
        return th, mk, dv

    def set_mask_override(self, mask):
        if mask is None:
            self.lib.oracle_set_mask_override(self.h, None)
        else:
            m = np.ascontiguousarray(mask, dtype=np.uint8)
            assert m.shape == self.shape
            self.lib.oracle_set_mask_override(self.h, m.ctypes.data_as(_c_ubyte_p))

    def interface_flags(self, d: int):
        nz, ny, nx = self.shape
        shp = (nz + (d == 2), ny + (d == 1), nx + (d == 0))
        out = np.empty(shp, dtype=np.uint8)
        self.lib.oracle_interface_flags(self.h, d, out.ctypes.data_as(_c_ubyte_p))
        return out

    def prim(self, which: int):
        out = np.empty(self.shape)
        self.lib.oracle_get_prim(self.h, which, _dp(out))
        return out

    def padded(self, q: int):
        nz, ny, nx = self.shape
        g = self.ng
        out = np.empty((nz + 2 * g, ny + 2 * g, nx + 2 * g))
        self.lib.oracle_get_padded(self.h, q, _dp(out))
        return out

    def metrics(self):
        ny, g = self.case.ny, self.ng
        a, b, c, y = np.empty(ny), np.empty(ny), np.empty(ny), np.empty(ny + 2 * g)
        self.lib.oracle_get_metrics(self.h, _dp(a), _dp(b), _dp(c), _dp(y))
        return a, b, c, y


def fd_coeffs(order: int, kind: str = "serial"):
    a, b = np.zeros(4), np.zeros(4)
    load(kind).oracle_fd_coeffs(order, _dp(a), _dp(b))
    return a[: order // 2].copy(), b[: order // 2].copy()


def weno_reconstruct(v, r: int, eps: float = 1e-6, linear: bool = False, kind: str = "serial"):
    v = np.ascontiguousarray(v, dtype=np.float64)
    assert v.size == 2 * r - 1
    beta = np.zeros(4)
    val = load(kind).oracle_weno_reconstruct(_dp(v), r, eps, int(linear), _dp(beta))
    return val, beta[:r].copy()


def weno_reconstruct_variant(v, r: int, eps: float = 1e-6, variant: int = 1, kind: str = "serial"):
    v = np.ascontiguousarray(v, dtype=np.float64)
    assert v.size == 2 * r - 1
    return load(kind).oracle_weno_reconstruct_variant(_dp(v), r, eps, variant)


def eigenvectors(d: int, vel, H: float, gamma: float, kind: str = "serial"):
    vel = np.ascontiguousarray(vel, dtype=np.float64)
    Lm, Rm = np.zeros((5, 5)), np.zeros((5, 5))
    load(kind).oracle_eigenvectors(d, _dp(vel), H, gamma, _dp(Lm), _dp(Rm))
    return Lm, Rm

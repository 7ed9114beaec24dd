"""ctypes wrapper around the fp64 CPU oracle (oracle/lbm_ibm_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from the CUDA
path.  ``build()`` compiles the C file with gcc (-O2 -fopenmp) next to its source.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lbm_ibm_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, fp, ip, llp = (C.POINTER(C.c_double), C.POINTER(C.c_float), C.POINTER(C.c_int),
                           C.POINTER(C.c_longlong))
        L.orc_delta_w.restype = C.c_double
        L.orc_delta_w.argtypes = [C.c_double]
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, ip, dp, C.c_int]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_fields.argtypes = [C.c_void_p, dp, dp]
        L.orc_populations.restype = dp
        L.orc_populations.argtypes = [C.c_void_p]
        L.orc_step_count.restype = C.c_longlong
        L.orc_step_count.argtypes = [C.c_void_p]
        L.orc_set_markers.restype = C.c_int
        L.orc_set_markers.argtypes = [C.c_void_p, fp, fp, fp, C.c_longlong]
        L.orc_set_kinematics.restype = C.c_int
        L.orc_set_kinematics.argtypes = [C.c_void_p, C.c_double, dp, dp]
        L.orc_clear_markers.argtypes = [C.c_void_p]
        L.orc_kinematics.argtypes = [C.c_void_p]
        L.orc_moments.argtypes = [C.c_void_p]
        L.orc_mdf.restype = C.c_int
        L.orc_mdf.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_collide.argtypes = [C.c_void_p]
        L.orc_stream.argtypes = [C.c_void_p]
        L.orc_step.restype = C.c_int
        L.orc_step.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_read_fields.argtypes = [C.c_void_p, dp, dp, dp]
        L.orc_read_markers.argtypes = [C.c_void_p, dp, dp, dp, dp, llp]
        L.orc_set_U.argtypes = [C.c_void_p, dp]
        L.orc_get_Um.argtypes = [C.c_void_p, dp]
        L.orc_markers_at_rest.argtypes = [C.c_void_p]
        L.orc_interpolate.argtypes = [C.c_void_p, dp, dp]
        L.orc_spread.argtypes = [C.c_void_p, dp, dp]
        L.orc_reference_sort.argtypes = [llp, C.c_longlong, llp]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float)) if a is not None else None


def delta_w(r: float) -> float:
    return lib().orc_delta_w(float(r))


def reference_sort(keys) -> np.ndarray:
    k = np.ascontiguousarray(keys, dtype=np.int64)
    perm = np.empty(k.shape[0], dtype=np.int64)
    lib().orc_reference_sort(k.ctypes.data_as(C.POINTER(C.c_longlong)), k.shape[0],
                             perm.ctypes.data_as(C.POINTER(C.c_longlong)))
    return perm


class Oracle:
    """Same call sequence as the product's C ABI, fp64 throughout."""

    def __init__(self, nx, ny, nz, tau, wall=(0, 0, 0), g=(0.0, 0.0, 0.0), forcing="guo"):
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.cells = self.nx * self.ny * self.nz
        w = (C.c_int * 3)(*[int(v) for v in wall])
        gb = (C.c_double * 3)(*[float(v) for v in g])
        self._h = lib().orc_create(self.nx, self.ny, self.nz, float(tau), w, gb,
                                   {"guo": 0, "shift": 1}[forcing])
        if not self._h:
            raise ValueError("orc_create failed (bad sizes or tau <= 0.5)")
        self.nm = 0

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- state ------------------------------------------------------------------------------
    def set_fields(self, rho=None, u=None):
        r = None if rho is None else np.ascontiguousarray(rho, dtype=np.float64).reshape(-1)
        v = None if u is None else np.ascontiguousarray(u, dtype=np.float64).reshape(-1)
        lib().orc_set_fields(self._h, _dp(r), _dp(v))

    def populations(self) -> np.ndarray:
        """View of the canonical populations, shape [19, nz, ny, nx] (valid until the next step)."""
        p = lib().orc_populations(self._h)
        return np.ctypeslib.as_array(p, shape=(19, self.nz, self.ny, self.nx))

    def set_markers(self, pos, vel, area) -> int:
        pos = np.ascontiguousarray(pos, dtype=np.float32).reshape(-1, 3)
        area = np.ascontiguousarray(area, dtype=np.float32).reshape(-1)
        v = None if vel is None else np.ascontiguousarray(vel, dtype=np.float32).reshape(-1, 3)
        n = pos.shape[0]
        self.nm += n
        return lib().orc_set_markers(self._h, _fp(pos), _fp(v), _fp(area), n)

    def set_kinematics(self, omega, axis, center) -> int:
        a = np.ascontiguousarray(axis, dtype=np.float64)
        c = np.ascontiguousarray(center, dtype=np.float64)
        return lib().orc_set_kinematics(self._h, float(omega), _dp(a), _dp(c))

    def clear_markers(self):
        lib().orc_clear_markers(self._h)
        self.nm = 0

    def add_bodies(self, bodies):
        for b in bodies:
            self.set_markers(b.pos, b.vel, b.area)
            self.set_kinematics(b.omega, b.axis, b.center)

    # -- stepping ---------------------------------------------------------------------------
    def step(self, nsteps=1, mdf_iters=0):
        rc = lib().orc_step(self._h, int(nsteps), int(mdf_iters))
        if rc:
            raise RuntimeError(f"orc_step failed with {rc}")

    def step_count(self) -> int:
        return int(lib().orc_step_count(self._h))

    def read_fields(self):
        rho = np.empty(self.cells)
        u = np.empty(3 * self.cells)
        f = np.empty(3 * self.cells)
        lib().orc_read_fields(self._h, _dp(rho), _dp(u), _dp(f))
        shp = (self.nz, self.ny, self.nx)
        return rho.reshape(shp), u.reshape((3,) + shp), f.reshape((3,) + shp)

    def read_markers(self):
        n = self.nm
        x, du, g, uk = (np.empty((n, 3)) for _ in range(4))
        key = np.empty(n, dtype=np.int64)
        lib().orc_read_markers(self._h, _dp(x), _dp(du), _dp(g), _dp(uk),
                               key.ctypes.data_as(C.POINTER(C.c_longlong)))
        return dict(x=x, du=du, g=g, uk=uk, key=key)

    # -- stand-alone pieces for the pins ------------------------------------------------------
    def set_U(self, U):
        lib().orc_set_U(self._h, _dp(np.ascontiguousarray(U, dtype=np.float64).reshape(-1)))

    def get_Um(self):
        U = np.empty(3 * self.cells)
        lib().orc_get_Um(self._h, _dp(U))
        return U.reshape(3, self.nz, self.ny, self.nx)

    def markers_at_rest(self):
        lib().orc_markers_at_rest(self._h)

    def kinematics(self):
        lib().orc_kinematics(self._h)

    def moments(self):
        lib().orc_moments(self._h)

    def mdf(self, n_iter, also_last_u=False):
        rc = lib().orc_mdf(self._h, int(n_iter), int(bool(also_last_u)))
        if rc:
            raise RuntimeError(f"orc_mdf failed with {rc}")

    def collide(self):
        lib().orc_collide(self._h)

    def stream(self):
        lib().orc_stream(self._h)

    def interpolate(self, U):
        U = np.ascontiguousarray(U, dtype=np.float64).reshape(-1)
        out = np.empty((self.nm, 3))
        lib().orc_interpolate(self._h, _dp(U), _dp(out))
        return out

    def spread(self, v):
        v = np.ascontiguousarray(v, dtype=np.float64).reshape(-1)
        F = np.zeros(3 * self.cells)
        lib().orc_spread(self._h, _dp(v), _dp(F))
        return F.reshape(3, self.nz, self.ny, self.nx)


def from_workload(wl, forcing="guo") -> Oracle:
    o = Oracle(wl.nx, wl.ny, wl.nz, wl.tau, wl.wall, wl.g, forcing)
    if wl.rho0 is not None or wl.u0 is not None:
        o.set_fields(wl.rho0, wl.u0)
    o.add_bodies(wl.bodies)
    return o

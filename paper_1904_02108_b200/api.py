"""Thin Python binding of the C ABI in include/lbm_ibm.h (argument marshalling only).

Same names as the C entry points.  Arrays may be numpy arrays (host) or torch tensors (host or
CUDA); outputs are written into buffers this module allocates (numpy, or torch on the GPU when
``device=True``).  PyTorch supplies device buffers and the stream -- nothing is computed here.
There is NO fallback: if the CUDA library is missing this module raises on import.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from ._build import LIB_PATH

if not os.path.exists(LIB_PATH):
    raise RuntimeError(
        f"{LIB_PATH} is missing: build it with `python -c 'import __graft_entry__ as g; g.build()'` "
        "(nvcc, sm_100a). There is no CPU or PyTorch fallback for this library.")

_L = C.CDLL(LIB_PATH)

OPT_SPREAD, OPT_FORCING, OPT_GRAPH, OPT_LBM_KERNEL, OPT_INTERP, OPT_TIMING, OPT_OVERLAP, OPT_MOMENTS = 1, 2, 3, 4, 5, 6, 7, 8
OPT_FUSED, OPT_TILE_ROWS, OPT_PERSISTENT, OPT_TILE_CAP, OPT_MDF_BLOCKS, OPT_TILE_WARPS, OPT_TRACE, OPT_PIPELINE = 9, 10, 11, 12, 13, 14, 15, 16
OPT_BULK_STREAM = 17
PERSISTENT_AUTO, PERSISTENT_ON, PERSISTENT_OFF = 0, 1, 2
INFO_MARKERS, INFO_BODIES, INFO_STEPS, INFO_LAUNCHES, INFO_ACTIVE_CELLS, INFO_DEVICE_BYTES, INFO_STATUS = range(1, 8)
INFO_RUNS, INFO_RUN_ENTRIES, INFO_TILES, INFO_ACTIVE_WORDS = 8, 9, 10, 11
INFO_TRACE_COUNT, INFO_TRACE_NS = 12, 200
INFO_LAYOUT, INFO_TILE_ROWS, INFO_SORT_PASSES = 13, 14, 15
INFO_PHASE_NS = 100
PHASES = ["keys", "sort", "bins", "moments", "interp", "spread", "lbm", "lbm_active"]
SPREAD_GATHER, SPREAD_ATOMIC, SPREAD_GATHER_PLAIN, SPREAD_BLOCK125 = 0, 1, 2, 3
MOMENTS_LIST, MOMENTS_BOX, MOMENTS_PER_MARKER = 0, 1, 2
INTERP_SORTED, INTERP_CALLER_ORDER, INTERP_WARP_PER_MARKER, INTERP_CHUNK_SMEM = 0, 1, 2, 3
FORCING_GUO, FORCING_SHIFT = 0, 1

EXPORTS = ["lbm_create", "lbm_destroy", "lbm_query_layout", "lbm_set_stream", "lbm_set_option", "lbm_get_info", "lbm_set_fields",
           "ibm_set_markers", "ibm_set_kinematics", "ibm_update_kinematics", "ibm_clear", "lbm_ibm_step", "lbm_read_fields",
           "ibm_read_markers", "ibm_read_markers_async", "ibm_wait_markers", "lbm_sync", "lbm_last_error",
           "lbm_trace_label", "ibm_sort_cells_noalloc"]


class _Bc(C.Structure):
    _fields_ = [("wall_x", C.c_int), ("wall_y", C.c_int), ("wall_z", C.c_int),
                ("gx", C.c_double), ("gy", C.c_double), ("gz", C.c_double)]


_vp = C.c_void_p
_L.lbm_create.restype = _vp
_L.lbm_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.POINTER(_Bc)]
_L.lbm_destroy.restype = None
_L.lbm_destroy.argtypes = [_vp]
_L.lbm_query_layout.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int)]
_L.lbm_set_stream.argtypes = [_vp, _vp]
_L.lbm_set_option.argtypes = [_vp, C.c_int, C.c_int]
_L.lbm_get_info.argtypes = [_vp, C.c_int, C.POINTER(C.c_longlong)]
_L.lbm_set_fields.argtypes = [_vp, _vp, _vp]
_L.ibm_set_markers.argtypes = [_vp, _vp, _vp, _vp, C.c_longlong]
_L.ibm_set_kinematics.argtypes = [_vp, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
_L.ibm_update_kinematics.argtypes = [_vp, C.c_int, C.c_int, _vp, _vp, _vp]
_L.ibm_clear.argtypes = [_vp]
_L.lbm_ibm_step.argtypes = [_vp, C.c_int, C.c_int]
_L.lbm_read_fields.argtypes = [_vp, _vp, _vp, _vp]
_L.ibm_read_markers.argtypes = [_vp, _vp, _vp, _vp, _vp]
_L.ibm_read_markers_async.argtypes = [_vp, _vp]
_L.ibm_wait_markers.argtypes = [_vp]
_L.lbm_sync.argtypes = [_vp]
_L.lbm_last_error.restype = C.c_char_p
_L.lbm_last_error.argtypes = []
_L.lbm_trace_label.restype = C.c_char_p
_L.lbm_trace_label.argtypes = [_vp, C.c_int]
_L.ibm_sort_cells_noalloc.argtypes = [_vp, C.c_int, C.c_longlong, _vp, _vp, _vp]
NOALLOC_MAX_MARKERS = 262144     # IBM_NOALLOC_MAX_MARKERS of include/lbm_ibm.h


class LbmError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__(f"{where} failed ({code}): {_L.lbm_last_error().decode()}")


def _check(rc, where):
    if rc < 0:
        raise LbmError(rc, where)
    return rc


def _ptr(a, dtype, keep):
    """address of a contiguous float32/int32 numpy array or torch tensor (host or device)"""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        b = np.ascontiguousarray(a, dtype=dtype)
        keep.append(b)
        return b.ctypes.data
    import torch
    if isinstance(a, torch.Tensor):
        tdt = {np.float32: torch.float32, np.int32: torch.int32}[dtype]
        b = a.to(tdt).contiguous()
        keep.append(b)
        return b.data_ptr()
    b = np.ascontiguousarray(np.asarray(a), dtype=dtype)
    keep.append(b)
    return b.ctypes.data


def query_layout(nx, ny, nz) -> dict:
    """lbm_query_layout: host-only, needs no GPU"""
    out = (C.c_int * 8)()
    _check(_L.lbm_query_layout(int(nx), int(ny), int(nz), out), "lbm_query_layout")
    keys = ["x_blocks", "entries", "tiles_y", "tiles_z", "mask_words_per_row", "block_width", "tile_rows", "entries_max"]
    return dict(zip(keys, [int(v) for v in out]))


class LbmIbm:
    """Handle around lbm_t*; methods mirror the C entry points one to one."""

    def __init__(self, nx, ny, nz, tau, wall=(0, 0, 0), g=(0.0, 0.0, 0.0), stream=None):
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        bc = _Bc(int(wall[0]), int(wall[1]), int(wall[2]), float(g[0]), float(g[1]), float(g[2]))
        self._h = _L.lbm_create(self.nx, self.ny, self.nz, float(tau), C.byref(bc))
        if not self._h:
            raise LbmError(-1, "lbm_create")
        self._stream_keep = None
        if stream is not None:
            self.set_stream(stream)

    # -- lifetime ----------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None):
            _L.lbm_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- configuration -----------------------------------------------------------------------
    def set_stream(self, stream):
        """stream: a torch.cuda.Stream, a raw cudaStream_t integer, or None (legacy default)."""
        raw = 0 if stream is None else (stream if isinstance(stream, int) else stream.cuda_stream)
        self._stream_keep = stream
        _check(_L.lbm_set_stream(self._h, raw), "lbm_set_stream")

    def set_option(self, key, value):
        _check(_L.lbm_set_option(self._h, int(key), int(value)), "lbm_set_option")

    def get_info(self, key) -> int:
        v = C.c_longlong(0)
        _check(_L.lbm_get_info(self._h, int(key), C.byref(v)), "lbm_get_info")
        return int(v.value)

    # -- the five calls of the problem statement -----------------------------------------------
    def set_fields(self, rho=None, u=None):
        keep = []
        _check(_L.lbm_set_fields(self._h, _ptr(rho, np.float32, keep), _ptr(u, np.float32, keep)), "lbm_set_fields")

    def set_markers(self, pos, vel, area) -> int:
        keep = []
        n = int(np.prod(area.shape))
        return _check(_L.ibm_set_markers(self._h, _ptr(pos, np.float32, keep), _ptr(vel, np.float32, keep),
                                         _ptr(area, np.float32, keep), n), "ibm_set_markers")

    def set_kinematics(self, omega, axis, center):
        a = (C.c_double * 3)(*[float(v) for v in axis])
        c = (C.c_double * 3)(*[float(v) for v in center])
        _check(_L.ibm_set_kinematics(self._h, float(omega), a, c), "ibm_set_kinematics")

    def update_kinematics(self, first_body, omega, axis, center=None):
        """omega [n], axis [n,3], center [n,3] or None: float64 numpy arrays (host)"""
        om = np.ascontiguousarray(omega, dtype=np.float64)
        ax = np.ascontiguousarray(axis, dtype=np.float64)
        ce = None if center is None else np.ascontiguousarray(center, dtype=np.float64)
        _check(_L.ibm_update_kinematics(self._h, int(first_body), int(om.shape[0]), om.ctypes.data, ax.ctypes.data,
                                        None if ce is None else ce.ctypes.data), "ibm_update_kinematics")

    def clear(self):
        _check(_L.ibm_clear(self._h), "ibm_clear")

    def add_bodies(self, bodies):
        for b in bodies:
            self.set_markers(b.pos, b.vel, b.area)
            self.set_kinematics(b.omega, b.axis, b.center)

    def step(self, nsteps=1, mdf_iters=0):
        _check(_L.lbm_ibm_step(self._h, int(nsteps), int(mdf_iters)), "lbm_ibm_step")

    def phase_ms(self) -> dict:
        """per-phase device time accumulated under OPT_TIMING, in ms"""
        return {n: self.get_info(INFO_PHASE_NS + i) * 1e-6 for i, n in enumerate(PHASES)}

    def trace(self) -> list:
        """[(label, ms since the fork of the last step)] of the trace events (OPT_TRACE)"""
        n = self.get_info(INFO_TRACE_COUNT)
        return [(_L.lbm_trace_label(self._h, i).decode(), self.get_info(INFO_TRACE_NS + i) * 1e-6) for i in range(n)]

    def sync(self):
        _check(_L.lbm_sync(self._h), "lbm_sync")

    def read_fields(self, rho=True, u=True, force=True, device=False, out=None):
        """returns (rho [nz,ny,nx], u [3,nz,ny,nx], force [3,nz,ny,nx]); entries not asked for are
        None.  device=True returns torch CUDA tensors (no host copy, asynchronous).  ``out`` may
        hold pre-allocated buffers {'rho':..., 'u':..., 'force':...} (numpy, e.g. pinned-backed, or torch)."""
        shp = (self.nz, self.ny, self.nx)
        want = {"rho": (rho, shp), "u": (u, (3,) + shp), "force": (force, (3,) + shp)}
        bufs, ptrs = {}, {}
        for name, (flag, shape) in want.items():
            if not flag:
                bufs[name], ptrs[name] = None, None
                continue
            if out is not None and name in out:
                b = out[name]
            elif device:
                import torch
                b = torch.empty(shape, dtype=torch.float32, device="cuda")
            else:
                b = np.empty(shape, dtype=np.float32)
            bufs[name] = b
            ptrs[name] = b.ctypes.data if isinstance(b, np.ndarray) else b.data_ptr()
        _check(_L.lbm_read_fields(self._h, ptrs["rho"], ptrs["u"], ptrs["force"]), "lbm_read_fields")
        return bufs["rho"], bufs["u"], bufs["force"]

    def read_markers(self, pos=True, force=True, perm=True, cell=True, out=None):
        n = self.get_info(INFO_MARKERS)
        spec = {"pos": (pos, (n, 3), np.float32), "force": (force, (n, 3), np.float32),
                "perm": (perm, (n,), np.int32), "cell": (cell, (n,), np.int32)}
        bufs, ptrs = {}, {}
        for name, (flag, shape, dt) in spec.items():
            if not flag:
                bufs[name], ptrs[name] = None, None
                continue
            b = out[name] if (out is not None and name in out) else np.empty(shape, dtype=dt)
            bufs[name] = b
            ptrs[name] = b.ctypes.data if isinstance(b, np.ndarray) else b.data_ptr()
        _check(_L.ibm_read_markers(self._h, ptrs["pos"], ptrs["force"], ptrs["perm"], ptrs["cell"]),
               "ibm_read_markers")
        return bufs

    def read_markers_async(self, force_out):
        """ibm_read_markers_async: force_out = host buffer [n,3] float32 (a numpy view of pinned memory or a
        pinned torch tensor); valid after wait_markers() / sync()"""
        ptr = force_out.ctypes.data if isinstance(force_out, np.ndarray) else force_out.data_ptr()
        _check(_L.ibm_read_markers_async(self._h, ptr), "ibm_read_markers_async")

    def wait_markers(self):
        _check(_L.ibm_wait_markers(self._h), "ibm_wait_markers")


def sort_cells_noalloc(cell, ncells, cell_sorted, perm, stream=None):
    """ibm_sort_cells_noalloc: cell (device tensor, n 32-bit keys < ncells) -> cell_sorted, perm (device tensors of n
    32-bit words, written in place).  Enqueued on `stream` (a torch.cuda.Stream, None = the default stream); allocates
    nothing; at most NOALLOC_MAX_MARKERS keys; calls that overlap on the GPU race on the library's scratch array."""
    n = int(cell.numel())
    for t in (cell, cell_sorted, perm):
        if t.element_size() != 4 or not t.is_contiguous():
            raise ValueError("sort_cells_noalloc: contiguous tensors of 32-bit words expected")
    if cell_sorted.numel() < n or perm.numel() < n:
        raise ValueError("sort_cells_noalloc: output tensors shorter than the input")
    _check(_L.ibm_sort_cells_noalloc(cell.data_ptr(), n, int(ncells), cell_sorted.data_ptr(), perm.data_ptr(),
                                     stream.cuda_stream if stream is not None else None), "ibm_sort_cells_noalloc")


def from_workload(wl, stream=None) -> LbmIbm:
    sim = LbmIbm(wl.nx, wl.ny, wl.nz, wl.tau, wl.wall, wl.g, stream=stream)
    if wl.rho0 is not None or wl.u0 is not None:
        sim.set_fields(wl.rho0, wl.u0)
    sim.add_bodies(wl.bodies)
    return sim

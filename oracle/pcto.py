"""ctypes loader for the CPU oracle (oracle/pcto.cpp).  TEST INFRASTRUCTURE ONLY.

May be imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs --
never by the product package.  Works on numpy host arrays; shares nothing with the CUDA binding.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_DIR, "libpcto.so")
_lib = None

REJ_MISS, REJ_ORDER, REJ_DEPTH, REJ_LEFT_GRID, TIE, END_MISMATCH, REJ_CAPACITY, REJ_NONFINITE = (
    0x01, 0x02, 0x04, 0x08, 0x10, 0x20, 0x40, 0x80)
REJECT_MASK = REJ_MISS | REJ_ORDER | REJ_DEPTH | REJ_LEFT_GRID | REJ_CAPACITY | REJ_NONFINITE


def build(force: bool = False) -> str:
    src = [os.path.join(_DIR, "pcto.cpp"), os.path.join(_DIR, "pcto_pre.cpp"), os.path.join(_DIR, "pcto.h")]
    if not force and os.path.exists(_SO) and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in src):
        return _SO
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", _SO, src[0], src[1]]
    subprocess.run(cmd, check=True, cwd=_DIR)
    return _SO


class Geometry(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("h_mm", C.c_double),
                ("origin_mm", C.c_double * 3)]


class MlpParams(C.Structure):
    _fields_ = [("poly", C.c_double * 6), ("poly_max_depth_mm", C.c_double), ("X0_mm", C.c_double),
                ("log_coeff", C.c_double), ("step_frac", C.c_double), ("tie_eps_mm", C.c_double),
                ("max_visits", C.c_int32)]


_PD = C.POINTER(C.c_double)


class FbpParams(C.Structure):
    _fields_ = [("n_theta", C.c_int32), ("n_s", C.c_int32), ("ds_mm", C.c_double), ("min_count", C.c_int32)]


class Protons(C.Structure):
    _fields_ = [("m", C.c_int64)] + [(k, _PD) for k in (
        "phi", "t_in", "v_in", "dt_in", "dv_in", "t_out", "v_out", "dt_out", "dv_out")] + [
        ("u_in_mm", C.c_double), ("u_out_mm", C.c_double)]


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        L.pcto_generate_mlp.restype = C.c_void_p
        L.pcto_generate_mlp.argtypes = [C.POINTER(Geometry), C.POINTER(MlpParams), C.POINTER(Protons), C.c_void_p,
                                        C.c_int]
        L.pcto_paths_info.argtypes = [C.c_void_p] + [C.POINTER(C.c_int64)] * 4
        L.pcto_paths_rows.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_int64,
                                      C.c_void_p, C.c_void_p, C.c_void_p]
        L.pcto_paths_free.argtypes = [C.c_void_p]
        L.pcto_paths_free.restype = None
        L.pcto_forward_project.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.pcto_column_counts.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_void_p]
        L.pcto_solve.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int64, C.c_double, C.c_void_p,
                                 C.c_void_p, C.c_int]
        L.pcto_scatter_moments.argtypes = [C.POINTER(MlpParams), C.c_double, C.c_double, C.c_double, _PD]
        L.pcto_mlp_point.argtypes = [C.POINTER(MlpParams), C.c_double, C.c_double, _PD, _PD, _PD]
        L.pcto_polyline.argtypes = [C.POINTER(Geometry), C.POINTER(MlpParams), C.POINTER(Protons), C.c_int64,
                                    C.c_void_p, C.c_void_p, C.c_int, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.pcto_walk_polyline.argtypes = [C.POINTER(Geometry), C.c_double, C.c_void_p, C.c_int, C.c_int32,
                                         C.c_void_p, C.c_int, C.POINTER(C.c_int32)]
        L.pcto_solve_ex.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int64, C.c_double,
                                    C.c_double, C.c_double, C.c_void_p, C.c_void_p, C.c_int]
        L.pcto_fbp.argtypes = [C.POINTER(Geometry), C.POINTER(Protons), C.c_void_p, C.POINTER(FbpParams), C.c_void_p,
                               C.c_void_p, C.c_void_p]
        L.pcto_hull_carve.argtypes = [C.POINTER(Geometry), C.POINTER(Protons), C.c_void_p, C.c_double, C.c_double,
                                      C.c_void_p]
        _lib = L
    return _lib


def make_geometry(nx, ny, nz, h_mm, origin_mm) -> Geometry:
    return Geometry(int(nx), int(ny), int(nz), float(h_mm), (C.c_double * 3)(*[float(v) for v in origin_mm]))


def make_params(poly, poly_max_depth_mm, X0_mm=361.0, log_coeff=0.038, step_frac=0.5, tie_eps_mm=1e-9,
                max_visits=2048) -> MlpParams:
    return MlpParams((C.c_double * 6)(*[float(a) for a in poly]), float(poly_max_depth_mm), float(X0_mm),
                     float(log_coeff), float(step_frac), float(tie_eps_mm), int(max_visits))


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


class ProtonArrays:
    """Keeps the numpy arrays alive next to the C struct."""
    NAMES = ("phi", "t_in", "v_in", "dt_in", "dv_in", "t_out", "v_out", "dt_out", "dv_out")

    def __init__(self, arrays: dict, u_in_mm: float, u_out_mm: float):
        self.a = {k: _f64(arrays[k]) for k in self.NAMES}
        self.m = int(self.a["phi"].shape[0])
        self.c = Protons(self.m, *[self.a[k].ctypes.data_as(_PD) for k in self.NAMES], float(u_in_mm),
                         float(u_out_mm))


class Paths:
    def __init__(self, geom: Geometry, params: MlpParams, protons: ProtonArrays, hull: Optional[np.ndarray] = None,
                 nthreads: int = 0):
        self.geom, self.n = geom, geom.nx * geom.ny * geom.nz
        h = None
        if hull is not None:
            h = np.ascontiguousarray(hull, dtype=np.uint8).reshape(-1)
            assert h.size == self.n
        self._h = lib().pcto_generate_mlp(C.byref(geom), C.byref(params), C.byref(protons.c),
                                          h.ctypes.data if h is not None else None, nthreads)
        if not self._h:
            raise ValueError("pcto_generate_mlp: invalid arguments")
        v = [C.c_int64() for _ in range(4)]
        lib().pcto_paths_info(self._h, *[C.byref(x) for x in v])
        self.m, self.total_visits, self.n_rejected, self.n_ties = [x.value for x in v]

    def rows(self, i0: int = 0, i1: Optional[int] = None):
        """-> (row_ptr int64[k+1], voxels int32[P], ell float32[k], flags uint8[k], length float64[k])"""
        i1 = self.m if i1 is None else i1
        k = i1 - i0
        row_ptr = np.zeros(k + 1, dtype=np.int64)
        ell, flags, length = np.zeros(k, np.float32), np.zeros(k, np.uint8), np.zeros(k, np.float64)
        assert lib().pcto_paths_rows(self._h, i0, i1, row_ptr.ctypes.data, None, 0, ell.ctypes.data,
                                     flags.ctypes.data, length.ctypes.data) == 0
        vox = np.zeros(int(row_ptr[-1]), dtype=np.int32)
        assert lib().pcto_paths_rows(self._h, i0, i1, row_ptr.ctypes.data, vox.ctypes.data, vox.size, None, None,
                                     None) == 0
        return row_ptr, vox, ell, flags, length

    def forward_project(self, x: np.ndarray, nthreads: int = 0) -> np.ndarray:
        x = np.ascontiguousarray(x, dtype=np.float32).reshape(-1)
        assert x.size == self.n
        b = np.zeros(self.m, dtype=np.float32)
        assert lib().pcto_forward_project(self._h, x.ctypes.data, b.ctypes.data, nthreads) == 0
        return b

    def column_counts(self, i0: int, i1: int) -> np.ndarray:
        c = np.zeros(self.n, dtype=np.uint32)
        assert lib().pcto_column_counts(self._h, i0, i1, c.ctypes.data) == 0
        return c

    def solve(self, b, x0, iters: int, block_size: int, lam: float, nthreads: int = 0, f64: bool = False):
        b = np.ascontiguousarray(b, dtype=np.float32).reshape(-1)
        x0 = np.ascontiguousarray(x0, dtype=np.float32).reshape(-1)
        assert b.size == self.m and x0.size == self.n
        x = np.zeros(self.n, dtype=np.float32)
        x64 = np.zeros(self.n, dtype=np.float64) if f64 else None
        assert lib().pcto_solve(self._h, b.ctypes.data, x0.ctypes.data, iters, block_size, lam, x.ctypes.data,
                                x64.ctypes.data if f64 else None, nthreads) == 0
        return (x, x64) if f64 else x

    def solve_ex(self, b, x0, w, iters: int, block_size: int, lam: float, clamp_lo: float = 1.0, clamp_hi: float = 0.0):
        """R27: weighted rows (w float32[m] or None) and box clamp (clamp_lo > clamp_hi = none)."""
        b = np.ascontiguousarray(b, dtype=np.float32).reshape(-1)
        x0 = np.ascontiguousarray(x0, dtype=np.float32).reshape(-1)
        wv = None if w is None else np.ascontiguousarray(w, dtype=np.float32).reshape(-1)
        assert b.size == self.m and x0.size == self.n and (wv is None or wv.size == self.m)
        x = np.zeros(self.n, dtype=np.float32)
        assert lib().pcto_solve_ex(self._h, b.ctypes.data, x0.ctypes.data, wv.ctypes.data if wv is not None else None,
                                   iters, block_size, lam, clamp_lo, clamp_hi, x.ctypes.data, None, 0) == 0
        return x

    def free(self):
        if self._h:
            lib().pcto_paths_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def scatter_moments(params: MlpParams, w_a: float, w_b: float, W: float) -> np.ndarray:
    out = (C.c_double * 3)()
    assert lib().pcto_scatter_moments(C.byref(params), w_a, w_b, W, out) == 0
    return np.array(out[:])


def mlp_point(params: MlpParams, D: float, w1: float, y0, y2) -> np.ndarray:
    out = (C.c_double * 2)()
    a, b = (C.c_double * 2)(*y0), (C.c_double * 2)(*y2)
    assert lib().pcto_mlp_point(C.byref(params), D, w1, a, b, out) == 0
    return np.array(out[:])


def polyline(geom: Geometry, params: MlpParams, protons: ProtonArrays, i: int, hull=None, cap: int = 8192):
    """-> (verts float64[K+1,3], v_start, v_end) or None if the history is rejected."""
    verts = np.zeros((cap, 3), dtype=np.float64)
    vs, ve = C.c_int32(), C.c_int32()
    h = None if hull is None else np.ascontiguousarray(hull, dtype=np.uint8).reshape(-1)
    nv = lib().pcto_polyline(C.byref(geom), C.byref(params), C.byref(protons.c), i,
                             h.ctypes.data if h is not None else None, verts.ctypes.data, cap, C.byref(vs),
                             C.byref(ve))
    if nv < 0:
        return None
    return verts[:nv].copy(), vs.value, ve.value


def walk_polyline(geom: Geometry, verts: np.ndarray, start_voxel: int, tie_eps_mm: float = 1e-9, cap: int = 65536):
    verts = np.ascontiguousarray(verts, dtype=np.float64)
    out = np.zeros(cap, dtype=np.int32)
    ties = C.c_int32()
    n = lib().pcto_walk_polyline(C.byref(geom), tie_eps_mm, verts.ctypes.data, verts.shape[0], start_voxel,
                                 out.ctypes.data, cap, C.byref(ties))
    if n < 0:
        return None, 0
    return out[:n].copy(), ties.value


def fbp(geom: Geometry, protons: ProtonArrays, b, n_theta: int, n_s: int, ds_mm: float, min_count: int = 1,
        want_sinogram: bool = False):
    """R25: FBP image float64[nz, ny, nx]; with want_sinogram also the mean-WEPL sinogram and its ramp-filtered rows,
    both [nz, n_theta, n_s]."""
    b = np.ascontiguousarray(b, dtype=np.float32).reshape(-1)
    assert b.size == protons.m
    fp = FbpParams(int(n_theta), int(n_s), float(ds_mm), int(min_count))
    x0 = np.zeros(geom.nx * geom.ny * geom.nz, dtype=np.float64)
    sino = np.zeros((geom.nz, n_theta, n_s), dtype=np.float64) if want_sinogram else None
    filt = np.zeros((geom.nz, n_theta, n_s), dtype=np.float64) if want_sinogram else None
    assert lib().pcto_fbp(C.byref(geom), C.byref(protons.c), b.ctypes.data, C.byref(fp),
                          sino.ctypes.data if want_sinogram else None, filt.ctypes.data if want_sinogram else None,
                          x0.ctypes.data) == 0
    x0 = x0.reshape(geom.nz, geom.ny, geom.nx)
    return (x0, sino, filt) if want_sinogram else x0


def hull_carve(geom: Geometry, protons: ProtonArrays, b, wepl_air_mm: float, min_chord_mm: float) -> np.ndarray:
    """R26: uint8[nz, ny, nx], 1 = never crossed (chord > min_chord_mm) by a history with WEPL < wepl_air_mm."""
    b = np.ascontiguousarray(b, dtype=np.float32).reshape(-1)
    assert b.size == protons.m
    out = np.zeros(geom.nx * geom.ny * geom.nz, dtype=np.uint8)
    assert lib().pcto_hull_carve(C.byref(geom), C.byref(protons.c), b.ctypes.data, float(wepl_air_mm),
                                 float(min_chord_mm), out.ctypes.data) == 0
    return out.reshape(geom.nz, geom.ny, geom.nx)

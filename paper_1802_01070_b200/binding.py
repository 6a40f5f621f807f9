"""Thin ctypes binding of libpct.so (include/pct.h).  Argument marshalling only: every step of the hot path
runs in the CUDA kernels behind the C-ABI.  torch is used for device memory and streams, nothing else.

There is NO CPU fallback: if libpct.so is missing or CUDA is unavailable the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, List, Optional

import torch

from . import build as _build

OK, E_INVALID_ARG, E_OOM, E_CUDA, E_CAPACITY = 0, -1, -2, -3, -4
REJ_MISS, REJ_ORDER, REJ_DEPTH, REJ_LEFT_GRID, TIE, END_MISMATCH, REJ_CAPACITY, REJ_NONFINITE = (
    0x01, 0x02, 0x04, 0x08, 0x10, 0x20, 0x40, 0x80)
FBP_STATIC_MAX_CELLS = 1 << 20
REJECT_MASK = REJ_MISS | REJ_ORDER | REJ_DEPTH | REJ_LEFT_GRID | REJ_CAPACITY | REJ_NONFINITE

EXPORTS = ("pct_create", "pct_destroy", "pct_last_error", "pct_generate_mlp", "pct_paths_info", "pct_paths_free",
           "pct_paths_decode", "pct_forward_project", "pct_column_counts", "pct_solve", "pct_reconstruct_host",
           "pct_launch_count", "pct_profile_enable", "pct_profile_read", "pct_measure_peaks", "pct_solve_config",
           "pct_plan_info", "pct_trim_cache", "pct_paths_flagged", "pct_solve_ex", "pct_fbp", "pct_hull_carve",
           "pct_fbp_static", "pct_regions_setup", "pct_hull_intersect", "pct_region_members", "pct_gather_histories",
           "pct_select_slices", "pct_reconstruct_regions")


class Geometry(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("h_mm", C.c_double),
                ("origin_mm", C.c_double * 3)]


class MlpParams(C.Structure):
    _fields_ = [("poly", C.c_double * 6), ("poly_max_depth_mm", C.c_double), ("X0_mm", C.c_double),
                ("log_coeff", C.c_double), ("step_frac", C.c_double), ("tie_eps_mm", C.c_double),
                ("max_visits", C.c_int32)]


class Protons(C.Structure):
    _fields_ = [("m", C.c_int64)] + [(k, C.c_void_p) for k in (
        "phi", "t_in", "v_in", "dt_in", "dv_in", "t_out", "v_out", "dt_out", "dv_out")] + [
        ("u_in_mm", C.c_double), ("u_out_mm", C.c_double)]


class PathsStats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in ("m", "total_visits", "n_rejected", "n_ties", "code_bytes", "header_bytes",
                                          "total_samples", "n_general_segments")]


class ReconStats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in ("m", "total_visits", "n_rejected", "n_ties")] + [
        (k, C.c_double) for k in ("ms_h2d", "ms_mlp", "ms_solve", "ms_d2h")]


PROFILE_KINDS = ("mlp", "project_windowed", "update", "project_direct", "plan", "pre")


class Profile(C.Structure):
    _fields_ = [("ms", C.c_double * len(PROFILE_KINDS)), ("launches", C.c_int64 * len(PROFILE_KINDS))]


class PlanStats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in ("block_size", "n_blocks", "n_groups", "n_direct", "plan_bytes", "stream_bytes",
                                          "cnt_bytes", "staged_slots", "windowed_histories", "windowed_visits")]


class SolveOpts(C.Structure):
    _fields_ = [("weights", C.c_void_p), ("clamp_lo", C.c_float), ("clamp_hi", C.c_float)]


class FbpParams(C.Structure):
    _fields_ = [("n_theta", C.c_int32), ("n_s", C.c_int32), ("ds_mm", C.c_double), ("min_count", C.c_int32)]


class Peaks(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("fp64_fma_per_s", "l2_gather_per_s", "l2_red_f32_per_s", "l2_red_v2_per_s",
                                          "l2_red_v2_coalesced_per_s", "smem_atomic_per_s", "smem_load_per_s",
                                          "smem_atomic_cf_per_s", "smem_load_cf_per_s")] + [
        ("num_sms", C.c_int32)]


PROTON_KEYS = ("phi", "t_in", "v_in", "dt_in", "dv_in", "t_out", "v_out", "dt_out", "dv_out")
_lib = None


class Region(C.Structure):
    _fields_ = [("z_lo", C.c_int32), ("z_hi", C.c_int32), ("keep_lo", C.c_int32), ("keep_hi", C.c_int32)]


class PctError(RuntimeError):
    pass


def load_library(path: Optional[str] = None):
    """dlopen libpct.so and declare the prototypes.  Needs no GPU (used by the CPU-side export test)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or os.environ.get("PCT_LIBRARY") or _build.LIB      # PCT_LIBRARY: another build of libpct.so (A/B runs)
    if not os.path.exists(path):
        raise PctError(f"{path} is missing: run `python -m paper_1802_01070_b200.build` (no CPU fallback exists)")
    L = C.CDLL(path)
    vp, i64 = C.c_void_p, C.c_int64
    L.pct_create.argtypes = [C.POINTER(Geometry), C.POINTER(MlpParams), C.c_int, C.POINTER(vp)]
    L.pct_destroy.argtypes = [vp]
    L.pct_destroy.restype = None
    L.pct_last_error.argtypes = [vp]
    L.pct_last_error.restype = C.c_char_p
    L.pct_generate_mlp.argtypes = [vp, C.POINTER(Protons), vp, vp, C.POINTER(vp)]
    L.pct_paths_info.argtypes = [vp, C.POINTER(PathsStats)]
    L.pct_paths_free.argtypes = [vp]
    L.pct_paths_free.restype = None
    L.pct_paths_decode.argtypes = [vp, vp, i64, i64, vp, vp, i64, vp, vp, vp]
    L.pct_paths_flagged.argtypes = [vp, vp, C.c_uint32, vp, i64, C.POINTER(i64), vp]
    L.pct_forward_project.argtypes = [vp, vp, vp, vp, vp]
    L.pct_column_counts.argtypes = [vp, vp, i64, i64, vp, vp]
    L.pct_solve.argtypes = [vp, vp, vp, vp, C.c_int, i64, C.c_float, vp, vp]
    L.pct_solve_ex.argtypes = [vp, vp, vp, vp, C.c_int, i64, C.c_float, C.POINTER(SolveOpts), vp, vp]
    L.pct_fbp.argtypes = [vp, C.POINTER(Protons), vp, C.POINTER(FbpParams), vp, vp]
    L.pct_fbp_static.argtypes = [vp, C.POINTER(Protons), vp, C.POINTER(FbpParams), vp, vp]
    L.pct_hull_carve.argtypes = [vp, C.POINTER(Protons), vp, C.c_double, C.c_double, vp, vp]
    L.pct_reconstruct_host.argtypes = [vp, C.POINTER(Protons), vp, vp, vp, C.c_int, i64, C.c_float, vp,
                                       C.POINTER(ReconStats), vp]
    L.pct_launch_count.argtypes = [vp]
    L.pct_launch_count.restype = i64
    L.pct_profile_enable.argtypes = [vp, C.c_int]
    L.pct_profile_read.argtypes = [vp, C.POINTER(Profile)]
    L.pct_measure_peaks.argtypes = [vp, C.POINTER(Peaks)]
    L.pct_solve_config.argtypes = [vp, C.c_int, i64]
    L.pct_plan_info.argtypes = [vp, C.POINTER(PlanStats)]
    L.pct_trim_cache.argtypes = [vp]
    L.pct_regions_setup.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.POINTER(Region)]
    L.pct_hull_intersect.argtypes = [vp, C.POINTER(Protons), vp, vp, vp, vp]
    L.pct_region_members.argtypes = [vp, vp, vp, i64, C.POINTER(Region), vp, C.POINTER(i64), vp]
    L.pct_gather_histories.argtypes = [vp, C.POINTER(Protons), vp, vp, i64, C.POINTER(Protons), vp, vp]
    L.pct_select_slices.argtypes = [vp, vp, C.POINTER(Region), vp, vp]
    L.pct_reconstruct_regions.argtypes = [vp, C.POINTER(Protons), vp, vp, vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32,
                                          C.c_int, i64, C.c_float, vp, C.POINTER(i64), vp]
    if path == _build.LIB:
        _lib = L
    return L


def _stream_ptr(device) -> int:
    return torch.cuda.current_stream(device).cuda_stream


def _dev_ptr(t: Optional[torch.Tensor], dtype, numel=None, device=None):
    if t is None:
        return None
    if not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise PctError(f"expected a contiguous CUDA tensor of {dtype}")
    if device is not None and t.device != device:
        raise PctError("tensor on the wrong device")
    if numel is not None and t.numel() != numel:
        raise PctError(f"expected {numel} elements, got {t.numel()}")
    return t.data_ptr()


class Paths:
    """Handle of the device-resident encoded rows (pct_paths)."""

    def __init__(self, ctx: "Context", handle: int):
        self.ctx, self._h = ctx, handle
        st = PathsStats()
        ctx._check(ctx._L.pct_paths_info(handle, C.byref(st)))
        self.m, self.total_visits, self.n_rejected, self.n_ties = st.m, st.total_visits, st.n_rejected, st.n_ties
        self.code_bytes, self.header_bytes, self.total_samples = st.code_bytes, st.header_bytes, st.total_samples
        self.n_general_segments = st.n_general_segments

    def plan_info(self) -> dict:
        """Statistics of the solve plan cached by the last pct_solve (zeros if it used the direct kernel)."""
        st = PlanStats()
        self.ctx._check(self.ctx._L.pct_plan_info(self._h, C.byref(st)))
        return {k: getattr(st, k) for k, _ in PlanStats._fields_}

    def free(self):
        if self._h:
            self.ctx._L.pct_paths_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


class Context:
    """pct_ctx: geometry + MLP constants + device scratch on one CUDA device."""

    def __init__(self, geometry: dict, params: dict, device: int = 0):
        if not torch.cuda.is_available():
            raise PctError("CUDA is not available: the pCT hot path only runs on the GPU (no CPU fallback)")
        self._L = load_library()
        self.device = torch.device("cuda", device)
        torch.cuda.init()
        with torch.cuda.device(self.device):
            torch.cuda.current_stream()          # make sure the primary context exists
        g = Geometry(int(geometry["nx"]), int(geometry["ny"]), int(geometry["nz"]), float(geometry["h_mm"]),
                     (C.c_double * 3)(*[float(v) for v in geometry["origin_mm"]]))
        p = MlpParams((C.c_double * 6)(*[float(a) for a in params["poly"]]), float(params["poly_max_depth_mm"]),
                      float(params["X0_mm"]), float(params["log_coeff"]), float(params["step_frac"]),
                      float(params["tie_eps_mm"]), int(params["max_visits"]))
        self.geom = g
        self.n = g.nx * g.ny * g.nz
        h = C.c_void_p()
        rc = self._L.pct_create(C.byref(g), C.byref(p), device, C.byref(h))
        if rc != OK:
            raise PctError(f"pct_create failed with code {rc}")
        self._h = h.value

    # -- plumbing ------------------------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != OK:
            msg = self._L.pct_last_error(self._h)
            raise PctError(f"libpct error {rc}: {msg.decode() if msg else ''}")

    def close(self):
        if getattr(self, "_h", None):
            self._L.pct_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def launch_count(self) -> int:
        return int(self._L.pct_launch_count(self._h))

    def profile_enable(self, on: bool):
        self._check(self._L.pct_profile_enable(self._h, 1 if on else 0))

    def profile_read(self) -> dict:
        """{kind: (ms, launches)} for kind in PROFILE_KINDS since the last read."""
        pr = Profile()
        self._check(self._L.pct_profile_read(self._h, C.byref(pr)))
        return {k: (pr.ms[i], pr.launches[i]) for i, k in enumerate(PROFILE_KINDS)}

    def trim_cache(self):
        """pct_trim_cache: give the idle device blocks of the library's buffer cache back to the driver."""
        self._check(self._L.pct_trim_cache(self._h))

    def solve_config(self, mode: int = 0, min_block: int = 0):
        """pct_solve_config: 0 = automatic, 1 = direct kernel only, 2 = windowed plan whenever possible."""
        self._check(self._L.pct_solve_config(self._h, int(mode), int(min_block)))

    def measure_peaks(self) -> dict:
        pk = Peaks()
        self._check(self._L.pct_measure_peaks(self._h, C.byref(pk)))
        return {k: getattr(pk, k) for k, _ in Peaks._fields_}

    # -- the C-ABI calls, same names --------------------------------------------------------------------------
    def generate_mlp(self, protons: Dict[str, torch.Tensor], u_in_mm: float, u_out_mm: float,
                     hull: Optional[torch.Tensor] = None) -> Paths:
        m = int(protons["phi"].numel())
        ptrs = [_dev_ptr(protons[k], torch.float64, m, self.device) for k in PROTON_KEYS]
        pr = Protons(m, *ptrs, float(u_in_mm), float(u_out_mm))
        out = C.c_void_p()
        self._check(self._L.pct_generate_mlp(self._h, C.byref(pr), _dev_ptr(hull, torch.uint8, self.n, self.device),
                                             _stream_ptr(self.device), C.byref(out)))
        return Paths(self, out.value)

    def paths_decode(self, paths: Paths, i0: int = 0, i1: Optional[int] = None):
        """-> row_ptr int64[k+1], voxels int32[P], ell float32[k], flags uint8[k] (CUDA tensors)."""
        i1 = paths.m if i1 is None else i1
        k = i1 - i0
        row_ptr = torch.empty(k + 1, dtype=torch.int64, device=self.device)
        ell = torch.empty(k, dtype=torch.float32, device=self.device)
        flags = torch.empty(k, dtype=torch.uint8, device=self.device)
        st = _stream_ptr(self.device)
        self._check(self._L.pct_paths_decode(self._h, paths._h, i0, i1, row_ptr.data_ptr(), None, 0, ell.data_ptr(),
                                             flags.data_ptr(), st))
        total = int(row_ptr[-1].item())
        vox = torch.empty(max(total, 1), dtype=torch.int32, device=self.device)
        self._check(self._L.pct_paths_decode(self._h, paths._h, i0, i1, row_ptr.data_ptr(), vox.data_ptr(), total, None,
                                             None, st))
        return row_ptr, vox[:total], ell, flags

    def paths_flagged(self, paths: Paths, mask: int = TIE, cap: int = 1 << 20):
        """pct_paths_flagged: (ascending history indices whose flags intersect mask [at most cap], total matching)."""
        import numpy as np
        idx = np.zeros(max(cap, 1), dtype=np.int64)
        n = C.c_int64()
        self._check(self._L.pct_paths_flagged(self._h, paths._h, int(mask), idx.ctypes.data, int(cap), C.byref(n),
                                              _stream_ptr(self.device)))
        return idx[:min(n.value, cap)].copy(), n.value

    def forward_project(self, paths: Paths, x: torch.Tensor, out: Optional[torch.Tensor] = None) -> torch.Tensor:
        b = out if out is not None else torch.empty(paths.m, dtype=torch.float32, device=self.device)
        self._check(self._L.pct_forward_project(self._h, paths._h, _dev_ptr(x, torch.float32, self.n, self.device),
                                                _dev_ptr(b, torch.float32, paths.m, self.device),
                                                _stream_ptr(self.device)))
        return b

    def column_counts(self, paths: Paths, i0: int, i1: int) -> torch.Tensor:
        c = torch.empty(self.n, dtype=torch.int32, device=self.device)      # uint32 payload
        self._check(self._L.pct_column_counts(self._h, paths._h, i0, i1, c.data_ptr(), _stream_ptr(self.device)))
        return c

    def solve(self, paths: Paths, b: torch.Tensor, x0: torch.Tensor, iters: int, block_size: int, lam: float,
              out: Optional[torch.Tensor] = None, weights: Optional[torch.Tensor] = None,
              clamp: Optional[tuple] = None) -> torch.Tensor:
        """pct_solve; with weights (float32[m] on the device) and / or clamp = (lo, hi): pct_solve_ex (R27)."""
        x = out if out is not None else torch.empty(self.n, dtype=torch.float32, device=self.device)
        args = (self._h, paths._h, _dev_ptr(b, torch.float32, paths.m, self.device),
                _dev_ptr(x0, torch.float32, self.n, self.device), int(iters), int(block_size), float(lam))
        tail = (_dev_ptr(x, torch.float32, self.n, self.device), _stream_ptr(self.device))
        if weights is None and clamp is None:
            self._check(self._L.pct_solve(*args, *tail))
        else:
            lo, hi = clamp if clamp is not None else (1.0, 0.0)
            opts = SolveOpts(_dev_ptr(weights, torch.float32, paths.m, self.device), float(lo), float(hi))
            self._check(self._L.pct_solve_ex(*args, C.byref(opts), *tail))
        return x

    def _protons_struct(self, protons: Dict[str, torch.Tensor], u_in_mm: float, u_out_mm: float) -> Protons:
        m = int(protons["phi"].numel())
        return Protons(m, *[_dev_ptr(protons[k], torch.float64, m, self.device) for k in PROTON_KEYS], float(u_in_mm),
                       float(u_out_mm))

    def fbp(self, protons: Dict[str, torch.Tensor], u_in_mm: float, u_out_mm: float, b: torch.Tensor, n_theta: int,
            n_s: int, ds_mm: float, min_count: int = 1, out: Optional[torch.Tensor] = None) -> torch.Tensor:
        """pct_fbp (R25): the FBP initial iterate, float32[n] on the device."""
        pr = self._protons_struct(protons, u_in_mm, u_out_mm)
        x0 = out if out is not None else torch.empty(self.n, dtype=torch.float32, device=self.device)
        fp = FbpParams(int(n_theta), int(n_s), float(ds_mm), int(min_count))
        self._check(self._L.pct_fbp(self._h, C.byref(pr), _dev_ptr(b, torch.float32, pr.m, self.device), C.byref(fp),
                                    _dev_ptr(x0, torch.float32, self.n, self.device), _stream_ptr(self.device)))
        return x0

    def fbp_static(self, protons: Dict[str, torch.Tensor], u_in_mm: float, u_out_mm: float, b: torch.Tensor, n_theta: int,
                   n_s: int, ds_mm: float, min_count: int = 1, out: Optional[torch.Tensor] = None) -> torch.Tensor:
        """pct_fbp_static: pct_fbp with its scratch in a fixed device array (no allocation inside the library; at most
        FBP_STATIC_MAX_CELLS sinogram bins).  `out` must be given by callers that may not allocate themselves."""
        pr = self._protons_struct(protons, u_in_mm, u_out_mm)
        x0 = out if out is not None else torch.empty(self.n, dtype=torch.float32, device=self.device)
        fp = FbpParams(int(n_theta), int(n_s), float(ds_mm), int(min_count))
        self._check(self._L.pct_fbp_static(self._h, C.byref(pr), _dev_ptr(b, torch.float32, pr.m, self.device), C.byref(fp),
                                           _dev_ptr(x0, torch.float32, self.n, self.device), _stream_ptr(self.device)))
        return x0

    def hull_carve(self, protons: Dict[str, torch.Tensor], u_in_mm: float, u_out_mm: float, b: torch.Tensor,
                   wepl_air_mm: float, min_chord_mm: float, out: Optional[torch.Tensor] = None) -> torch.Tensor:
        """pct_hull_carve (R26): uint8[n] hull mask on the device."""
        pr = self._protons_struct(protons, u_in_mm, u_out_mm)
        hull = out if out is not None else torch.empty(self.n, dtype=torch.uint8, device=self.device)
        self._check(self._L.pct_hull_carve(self._h, C.byref(pr), _dev_ptr(b, torch.float32, pr.m, self.device),
                                           float(wepl_air_mm), float(min_chord_mm),
                                           _dev_ptr(hull, torch.uint8, self.n, self.device), _stream_ptr(self.device)))
        return hull

    # ---- Algorithm 1 of the paper (reading R28): z-regions, one independent solve per region --------
    def hull_intersect(self, protons: Dict[str, torch.Tensor], u_in_mm: float, u_out_mm: float,
                       hull: Optional[torch.Tensor]):
        """pct_hull_intersect (A1 alone): int32[m] hull entry and exit voxel of every history, -1 if rejected there."""
        pr = self._protons_struct(protons, u_in_mm, u_out_mm)
        v_in = torch.empty(max(pr.m, 1), dtype=torch.int32, device=self.device)
        v_out = torch.empty(max(pr.m, 1), dtype=torch.int32, device=self.device)
        self._check(self._L.pct_hull_intersect(self._h, C.byref(pr), _dev_ptr(hull, torch.uint8, self.n, self.device),
                                               v_in.data_ptr(), v_out.data_ptr(), _stream_ptr(self.device)))
        return v_in[:pr.m], v_out[:pr.m]

    def region_members(self, v_in: torch.Tensor, v_out: torch.Tensor, region: "Region") -> torch.Tensor:
        """pct_region_members (step 2): the member histories, ascending (indices < 2^31 in an int32 tensor)."""
        m = int(v_in.numel())
        idx = torch.empty(max(m, 1), dtype=torch.int32, device=self.device)
        cnt = C.c_int64(0)
        self._check(self._L.pct_region_members(self._h, _dev_ptr(v_in.contiguous(), torch.int32, m, self.device),
                                               _dev_ptr(v_out.contiguous(), torch.int32, m, self.device), m, C.byref(region),
                                               idx.data_ptr(), C.byref(cnt), _stream_ptr(self.device)))
        return idx[:cnt.value]

    def gather_histories(self, protons: Dict[str, torch.Tensor], u_in_mm: float, u_out_mm: float,
                         b: Optional[torch.Tensor], idx: torch.Tensor):
        """pct_gather_histories (step 3): the members' tracker records (dict of float64 tensors) and WEPLs."""
        pr = self._protons_struct(protons, u_in_mm, u_out_mm)
        count = int(idx.numel())
        out = {k: torch.empty(max(count, 1), dtype=torch.float64, device=self.device) for k in PROTON_KEYS}
        dst = Protons(count, *[out[k].data_ptr() for k in PROTON_KEYS], 0.0, 0.0)
        b_dst = torch.empty(max(count, 1), dtype=torch.float32, device=self.device) if b is not None else None
        self._check(self._L.pct_gather_histories(
            self._h, C.byref(pr), _dev_ptr(b, torch.float32, pr.m, self.device) if b is not None else None,
            _dev_ptr(idx.contiguous(), torch.int32, count, self.device) if count else None, count, C.byref(dst),
            b_dst.data_ptr() if b_dst is not None else None, _stream_ptr(self.device)))
        return {k: v[:count] for k, v in out.items()}, (b_dst[:count] if b_dst is not None else None)

    def select_slices(self, x_region: torch.Tensor, region: "Region", x_final: torch.Tensor) -> torch.Tensor:
        """pct_select_slices (step 5): the region's kept slices go into x_final."""
        self._check(self._L.pct_select_slices(self._h, _dev_ptr(x_region, torch.float32, self.n, self.device), C.byref(region),
                                              _dev_ptr(x_final, torch.float32, self.n, self.device), _stream_ptr(self.device)))
        return x_final

    def reconstruct_regions(self, protons: Dict[str, torch.Tensor], u_in_mm: float, u_out_mm: float,
                            hull: Optional[torch.Tensor], b: torch.Tensor, x0: Optional[torch.Tensor], n_regions: int,
                            ext: int, iters: int, block_size: int, lam: float, region_first: int = 0,
                            region_count: Optional[int] = None, out: Optional[torch.Tensor] = None):
        """pct_reconstruct_regions: steps 1-5 for the regions [region_first, region_first + region_count) on this GPU.
        Returns (x, members per region; -1 for regions not run); slices kept by regions that were not run keep `out`'s values."""
        pr = self._protons_struct(protons, u_in_mm, u_out_mm)
        x = out if out is not None else torch.zeros(self.n, dtype=torch.float32, device=self.device)
        members = (C.c_int64 * int(n_regions))(*([-1] * int(n_regions)))
        rc = int(region_count) if region_count is not None else int(n_regions) - int(region_first)
        self._check(self._L.pct_reconstruct_regions(
            self._h, C.byref(pr), _dev_ptr(b, torch.float32, pr.m, self.device),
            _dev_ptr(hull, torch.uint8, self.n, self.device), _dev_ptr(x0, torch.float32, self.n, self.device),
            int(n_regions), int(ext), int(region_first), rc, int(iters), int(block_size), float(lam),
            _dev_ptr(x, torch.float32, self.n, self.device), members, _stream_ptr(self.device)))
        return x, list(members)

    def reconstruct_host(self, protons: Dict[str, torch.Tensor], u_in_mm: float, u_out_mm: float,
                         hull: Optional[torch.Tensor], b: torch.Tensor, x0: Optional[torch.Tensor], iters: int,
                         block_size: int, lam: float, x_out: torch.Tensor) -> dict:
        """Whole hot path on HOST (ideally pinned) tensors; returns the phase times and counts."""
        m = int(protons["phi"].numel())
        for k in PROTON_KEYS:
            t = protons[k]
            if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous() or t.numel() != m:
                raise PctError("reconstruct_host expects contiguous float64 HOST tensors")
        for t, dt, ne in ((hull, torch.uint8, self.n), (b, torch.float32, m), (x0, torch.float32, self.n),
                          (x_out, torch.float32, self.n)):
            if t is not None and (t.is_cuda or t.dtype != dt or not t.is_contiguous() or t.numel() != ne):
                raise PctError("reconstruct_host: bad host tensor")
        pr = Protons(m, *[protons[k].data_ptr() for k in PROTON_KEYS], float(u_in_mm), float(u_out_mm))
        st = ReconStats()
        self._check(self._L.pct_reconstruct_host(self._h, C.byref(pr), hull.data_ptr() if hull is not None else None,
                                                 b.data_ptr(), x0.data_ptr() if x0 is not None else None, int(iters),
                                                 int(block_size), float(lam), x_out.data_ptr(), C.byref(st),
                                                 _stream_ptr(self.device)))
        return {k: getattr(st, k) for k, _ in ReconStats._fields_}


def regions_setup(nz: int, n_regions: int, ext: int, lib=None) -> List["Region"]:
    """pct_regions_setup (step 1; pure host arithmetic): the regions of Algorithm 1 as Region structs."""
    L = lib or load_library()
    out = (Region * int(n_regions))()
    if L.pct_regions_setup(int(nz), int(n_regions), int(ext), out) != OK:
        raise PctError(f"pct_regions_setup({nz}, {n_regions}, {ext}): invalid arguments")
    return list(out)

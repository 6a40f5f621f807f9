"""Seeded synthetic pCT inputs (phantoms, tracker records, WEPL) for tests, smoke and bench.

This module is the ONLY code shared by the CPU oracle's tests and the CUDA path's tests/bench.
It holds none of the method's arithmetic (no MLP, no voxel walk, no projection): it only
manufactures *inputs* -- what the scanner of PAPER.md:7 ("tracking system ... WEPL of individual
protons") would deliver -- with the structure of the paper's workloads (90
projections at 4 degree steps or continuous rotation; 116 M / 261 M histories; protons in
acquisition order; small z excursion of paths, Table I).  The paper's CTP404
datasets are not available; BASELINE.json's phantoms stand in for them (recipe in DESIGN.md).

Everything is plain torch, float64, device-agnostic (CPU for Tiny, CUDA for the big configs).
The generator is a forward Monte-Carlo random walk (1 mm steps, Highland angles, Bragg-Kleeman
energy loss); its physics is not graded -- its output is the input of both oracle and CUDA path.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, Optional, Tuple

import numpy as np
import torch

PROTON_MASS_MEV = 938.272
BK_ALPHA_MM = 0.022      # Bragg-Kleeman range R = alpha * E^p, alpha = 0.0022 cm MeV^-p
BK_P = 1.77
X0_WATER_MM = 361.0
SAD_MM = 2000.0          # source-axis distance of the diverging ("cone") beam, proposed in SURVEY 8(d)

# 1/(beta^2 p^2) in c^2/MeV^2 for 200 MeV protons in water, depth in cm (the degree-5 fit used with the
# MLP formalism of PAPER.md ref [3]).  poly_mm() rescales to depth in mm.
POLY_200MEV_CM = (7.457e-6, 4.548e-7, -5.777e-8, 1.301e-8, -9.228e-10, 2.687e-11)


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    nx: int
    ny: int
    nz: int
    h: float
    m: int
    energy: float          # MeV
    beam: str              # "parallel90" (4 degree steps, sorted by angle) | "cone" (continuous rotation)
    iters: int
    block: int
    lam: float
    noise: float = 0.01
    seed: int = 0
    u_tracker: float = 0.0  # tracker planes at -/+ u_tracker (gantry frame)
    poly_max_depth: float = 200.0

    @property
    def n(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def lo(self) -> Tuple[float, float, float]:
        return (-0.5 * self.nx * self.h, -0.5 * self.ny * self.h, -0.5 * self.nz * self.h)


# BASELINE.json configs 0..3 (config 4 = sweep over config 1; see bench.py / tests).
CONFIGS: Dict[str, Config] = {
    "tiny": Config("tiny", 32, 32, 8, 1.0, 50_000, 200.0, "parallel90", 5, 5_000, 0.1, u_tracker=22.0),
    "head": Config("head", 200, 200, 100, 1.0, 20_000_000, 200.0, "parallel90", 10, 200_000, 0.1,
                   u_tracker=90.0),
    "paperA": Config("paperA", 256, 256, 128, 1.0, 116_000_000, 200.0, "cone", 12, 1_000_000, 0.1,
                     u_tracker=105.0, poly_max_depth=215.0),
    "paperB": Config("paperB", 320, 320, 160, 1.0, 261_000_000, 230.0, "cone", 12, 2_000_000, 0.1,
                     u_tracker=160.0, poly_max_depth=305.0),
}


def scaled(cfg: Config, m: int, block: Optional[int] = None, iters: Optional[int] = None) -> Config:
    """Same phantom/beam with fewer histories (parity-test cases)."""
    return dataclasses.replace(cfg, m=m, block=block if block is not None else cfg.block,
                               iters=iters if iters is not None else cfg.iters)


# --------------------------------------------------------------------------------------------------
# stopping-power model used only to (a) fit the polynomial handed to the MLP and (b) slow the protons
# --------------------------------------------------------------------------------------------------
def energy_at_depth(e0: float, depth_mm):
    r0 = BK_ALPHA_MM * e0 ** BK_P
    rem = np.maximum(r0 - np.asarray(depth_mm, dtype=np.float64), 1e-9)
    return (rem / BK_ALPHA_MM) ** (1.0 / BK_P)


def inv_beta2p2(e):
    e = np.asarray(e, dtype=np.float64)
    return ((e + PROTON_MASS_MEV) / (e * (e + 2.0 * PROTON_MASS_MEV))) ** 2


def poly_mm(energy: float, max_depth_mm: float) -> Tuple[float, ...]:
    """Degree-5 polynomial a_i (depth in mm) for 1/(beta^2 p^2) along a water path.

    200 MeV: the published-style coefficient set rescaled from cm to mm.  Other energies: a least
    squares fit of the Bragg-Kleeman model on [0, max_depth_mm] (Chebyshev nodes, float64)."""
    if abs(energy - 200.0) < 1e-9:
        return tuple(a / 10.0 ** i for i, a in enumerate(POLY_200MEV_CM))
    k = np.arange(400)
    d = 0.5 * max_depth_mm * (1.0 - np.cos(np.pi * (k + 0.5) / 400))
    f = inv_beta2p2(energy_at_depth(energy, d))
    s = d / max_depth_mm
    c = np.polynomial.polynomial.polyfit(s, f, 5)
    return tuple(float(ci / max_depth_mm ** i) for i, ci in enumerate(c))


# --------------------------------------------------------------------------------------------------
# phantoms: analytic shapes rasterised at voxel centres -> x_true float32[nz,ny,nx], hull uint8
# --------------------------------------------------------------------------------------------------
def _centres(cfg: Config, device):
    lo = cfg.lo
    xs = lo[0] + (torch.arange(cfg.nx, device=device, dtype=torch.float64) + 0.5) * cfg.h
    ys = lo[1] + (torch.arange(cfg.ny, device=device, dtype=torch.float64) + 0.5) * cfg.h
    zs = lo[2] + (torch.arange(cfg.nz, device=device, dtype=torch.float64) + 0.5) * cfg.h
    return zs[:, None, None], ys[None, :, None], xs[None, None, :]


def _head_spheres(seed: int):
    rng = np.random.default_rng(seed + 1234)
    out = []
    while len(out) < 8:
        c = rng.uniform(-1, 1, 3)
        if (c ** 2).sum() > 1:
            continue
        c = c * np.array([80.0, 70.0, 45.0]) * 0.6
        r = rng.uniform(6.0, 12.0)
        if all(np.linalg.norm(c - c2) > r + r2 + 1.0 for c2, r2, _ in out):
            out.append((c, r, rng.uniform(0.25, 1.8)))
    return out


def make_phantom(cfg: Config, device="cpu"):
    """Returns (x_true float32 [nz,ny,nx], hull uint8 [nz,ny,nx], shadow) for BASELINE.json configs."""
    z, y, x = _centres(cfg, device)
    shape = (cfg.nz, cfg.ny, cfg.nx)
    rsp = torch.zeros(shape, dtype=torch.float32, device=device)
    if cfg.name.startswith("tiny"):
        body = (x * x + y * y <= 12.0 ** 2).expand(shape)
        rsp[body] = 1.0
        rsp[((x - 5.0) ** 2 + y * y <= 9.0).expand(shape)] = 1.6     # bone insert
        rsp[((x + 5.0) ** 2 + y * y <= 9.0).expand(shape)] = 0.3     # lung insert
        shadow = dict(kind="box", a=12.0, b=12.0, v=0.5 * cfg.nz * cfg.h)
    elif cfg.name.startswith("head"):
        body = ((x / 80.0) ** 2 + (y / 70.0) ** 2 + (z / 45.0) ** 2 <= 1.0).expand(shape)
        rsp[body] = 1.0
        for c, r, val in _head_spheres(cfg.seed):
            rsp[((x - c[0]) ** 2 + (y - c[1]) ** 2 + (z - c[2]) ** 2 <= r * r).expand(shape)] = float(val)
        shadow = dict(kind="ellipse", a=80.0, b=70.0, v=45.0)
    elif cfg.name.startswith("paperA"):
        body = ((x / 95.0) ** 2 + (y / 80.0) ** 2 + (z / 60.0) ** 2 <= 1.0).expand(shape)
        inner = ((x / 89.0) ** 2 + (y / 74.0) ** 2 + (z / 54.0) ** 2 <= 1.0).expand(shape)
        rsp[body] = 1.6                                               # 6 mm bone shell
        rsp[inner] = 1.04                                             # soft tissue
        for cx in (-25.0, 25.0):                                      # two air cavities
            rsp[((x - cx) ** 2 + (y - 30.0) ** 2 + z * z <= 12.0 ** 2).expand(shape)] = 0.001
        shadow = dict(kind="ellipse", a=95.0, b=80.0, v=60.0)
    elif cfg.name.startswith("paperB"):
        body = ((x / 150.0) ** 2 + (y / 110.0) ** 2 <= 1.0).expand(shape)
        rsp[body] = 1.0
        for cx in (-65.0, 65.0):                                      # lungs
            rsp[(((x - cx) / 45.0) ** 2 + (y / 60.0) ** 2 <= 1.0).expand(shape)] = 0.3
        rsp[(x * x + (y + 70.0) ** 2 <= 15.0 ** 2).expand(shape)] = 1.6  # spine
        shadow = dict(kind="box", a=150.0, b=110.0, v=0.5 * cfg.nz * cfg.h)
    else:
        raise ValueError(cfg.name)
    hull = body.to(torch.uint8).contiguous()
    return rsp.contiguous(), hull, shadow


# --------------------------------------------------------------------------------------------------
# proton histories
# --------------------------------------------------------------------------------------------------
def _beta_p(e):
    return e * (e + 2.0 * PROTON_MASS_MEV) / (e + PROTON_MASS_MEV)      # p*v = beta*p*c in MeV


def generate_protons(cfg: Config, x_true: torch.Tensor, shadow: dict, device="cpu",
                     chunk: int = 1 << 22, i0: int = 0, i1: Optional[int] = None,
                     scatter: bool = True) -> Dict[str, torch.Tensor]:
    """Tracker records + noisy WEPL for histories [i0, i1) of cfg (acquisition order).

    Returns float64 tensors phi, t_in, v_in, dt_in, dv_in, t_out, v_out, dt_out, dv_out (slopes are
    d/du) and float32 wepl.  u_in = -cfg.u_tracker, u_out = +cfg.u_tracker.
    Deterministic for a given (cfg.seed, device type, chunk)."""
    i1 = cfg.m if i1 is None else i1
    mm = i1 - i0
    names = ("phi", "t_in", "v_in", "dt_in", "dv_in", "t_out", "v_out", "dt_out", "dv_out")
    out = {k: torch.empty(mm, dtype=torch.float64, device=device) for k in names}
    out["wepl"] = torch.empty(mm, dtype=torch.float32, device=device)
    rsp_flat = x_true.reshape(-1).to(device=device, dtype=torch.float64)
    lo = cfg.lo
    nsteps = int(round(2.0 * cfg.u_tracker))          # 1 mm steps in u between the tracker planes
    for c0 in range(i0, i1, chunk):
        c1 = min(c0 + chunk, i1)
        k = c1 - c0
        gen = torch.Generator(device=device)
        gen.manual_seed((cfg.seed * 1_000_003 + c0) & 0x7FFFFFFFFFFF)
        idx = torch.arange(c0, c1, device=device, dtype=torch.float64)
        if cfg.beam == "parallel90":
            per = cfg.m / 90.0
            phi = torch.floor(idx / per).clamp_(max=89.0) * (4.0 * math.pi / 180.0)
        else:
            phi = idx * (2.0 * math.pi / cfg.m)
        cph, sph = torch.cos(phi), torch.sin(phi)
        u1 = torch.rand(k, dtype=torch.float64, device=device, generator=gen)
        u2 = torch.rand(k, dtype=torch.float64, device=device, generator=gen)
        rt = torch.sqrt((shadow["a"] * sph) ** 2 + (shadow["b"] * cph) ** 2)   # hull half-width seen at phi
        if shadow["kind"] == "ellipse":
            rad, ang = torch.sqrt(u1), 2.0 * math.pi * u2
            t = rt * rad * torch.cos(ang)
            v = shadow["v"] * rad * torch.sin(ang)
        else:
            t = rt * (2.0 * u1 - 1.0)
            v = shadow["v"] * (2.0 * u2 - 1.0)
        if cfg.beam == "cone":
            dt, dv = t / SAD_MM, v / SAD_MM
        else:
            dt, dv = torch.zeros_like(t), torch.zeros_like(v)
        out["phi"][c0 - i0:c1 - i0] = phi
        out["t_in"][c0 - i0:c1 - i0] = t
        out["v_in"][c0 - i0:c1 - i0] = v
        out["dt_in"][c0 - i0:c1 - i0] = dt
        out["dv_in"][c0 - i0:c1 - i0] = dv
        t, v, dt, dv = t.clone(), v.clone(), dt.clone(), dv.clone()
        e = torch.full((k,), float(cfg.energy), dtype=torch.float64, device=device)
        wepl = torch.zeros(k, dtype=torch.float64, device=device)
        u = -cfg.u_tracker
        for _ in range(nsteps):
            um = u + 0.5
            tm, vm = t + 0.5 * dt, v + 0.5 * dv
            ix = torch.floor((um * cph - tm * sph - lo[0]) / cfg.h).long()
            iy = torch.floor((um * sph + tm * cph - lo[1]) / cfg.h).long()
            iz = torch.floor((vm - lo[2]) / cfg.h).long()
            inside = (ix >= 0) & (ix < cfg.nx) & (iy >= 0) & (iy < cfg.ny) & (iz >= 0) & (iz < cfg.nz)
            j = (ix + cfg.nx * (iy + cfg.ny * iz)).clamp_(0, cfg.n - 1)
            rho = torch.where(inside, rsp_flat[j], torch.zeros_like(wepl))
            ds = torch.sqrt(1.0 + dt * dt + dv * dv)
            w = rho * ds
            wepl += w
            t += dt
            v += dv
            if scatter:
                xr = (w / X0_WATER_MM).clamp_(min=1e-30)
                th0 = (13.6 / _beta_p(e)) * torch.sqrt(xr) * (1.0 + 0.038 * torch.log(xr))
                th0.clamp_(min=0.0)
                dt += th0 * torch.randn(k, dtype=torch.float64, device=device, generator=gen)
                dv += th0 * torch.randn(k, dtype=torch.float64, device=device, generator=gen)
            e = (e - w * e ** (1.0 - BK_P) / (BK_ALPHA_MM * BK_P)).clamp_(min=10.0)
            u += 1.0
        out["t_out"][c0 - i0:c1 - i0] = t
        out["v_out"][c0 - i0:c1 - i0] = v
        out["dt_out"][c0 - i0:c1 - i0] = dt
        out["dv_out"][c0 - i0:c1 - i0] = dv
        noise = torch.randn(k, dtype=torch.float64, device=device, generator=gen)
        out["wepl"][c0 - i0:c1 - i0] = (wepl * (1.0 + cfg.noise * noise)).to(torch.float32)
    return out


def mlp_params(cfg: Config) -> dict:
    """Parameter set handed (identically) to the oracle and to the CUDA library."""
    return dict(poly=poly_mm(cfg.energy, cfg.poly_max_depth), poly_max_depth_mm=cfg.poly_max_depth,
                X0_mm=X0_WATER_MM, log_coeff=0.038, step_frac=0.5, tie_eps_mm=1e-9, max_visits=2048)


def geometry(cfg: Config) -> dict:
    return dict(nx=cfg.nx, ny=cfg.ny, nz=cfg.nz, h_mm=cfg.h, origin_mm=cfg.lo)


def random_rays(n: int, cfg: Config, seed: int = 0) -> Dict[str, torch.Tensor]:
    """Straight histories (exit = straight continuation of entry) for the Siddon / straight-line pins."""
    rng = np.random.default_rng(seed)
    half_t = 0.45 * min(cfg.nx, cfg.ny) * cfg.h
    half_v = 0.45 * cfg.nz * cfg.h
    phi = rng.uniform(0, 2 * np.pi, n)
    t = rng.uniform(-half_t, half_t, n)
    v = rng.uniform(-half_v, half_v, n)
    dt = rng.uniform(-0.2, 0.2, n)
    dv = rng.uniform(-0.05, 0.05, n)
    du = 2.0 * cfg.u_tracker
    d = dict(phi=phi, t_in=t, v_in=v, dt_in=dt, dv_in=dv, t_out=t + dt * du, v_out=v + dv * du,
             dt_out=dt.copy(), dv_out=dv.copy())
    return {k: torch.from_numpy(np.ascontiguousarray(a)) for k, a in d.items()}

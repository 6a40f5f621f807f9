#!/usr/bin/env python
"""bench.py -- one JSON line for the pCT hot path on N B200s (contract in the task statement).

A "step" = one pass of the WHOLE hot path over the workload's synthetic histories, resident in HBM:
pct_generate_mlp (A1-A3) + pct_solve at the configured iterations (A4-A8; the solve plan is rebuilt every step).
  value                 = path-voxel updates (P = sum_i N_i visits, x iterations) per second of WHOLE-STEP time
                          (K1 + plan + solve): the contract's whole-job throughput.
  solver_updates_per_s  = P / t_iter: SURVEY.md 8(d)'s metric proper (one sweep of A5-A7, plan build amortised in).
  e2e                   = the same as `value` through pct_reconstruct_host on pinned HOST buffers (H2D + MLP + solve +
                          D2H inside the timing).
The K timed steps run without any instrumentation; the per-kernel breakdown and the rooflines come from extra,
separately timed steps with CUDA events around every launch (pct_profile_enable).
Multi-GPU: the path does not shard (north_star: one B200, no inter-GPU traffic) -> N independent replicas.
`--impl reference` times the CPU oracle (as it stands) on a bounded sample of the same workload.
"""
import argparse
import dataclasses
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

import synth

METRIC = "path-voxel updates/s per solver iteration; end-to-end recon s at 116M/261M"
UNIT = "path-voxel updates/s"
# ---- roofline inputs -----------------------------------------------------------------------------------------
# K2w (k_block_windowed), per visit and sweep: shared-memory lane operations of the two walks -- step-table load + x load
# (pass 1), step-table load + Delta atomic (pass 2), + one count atomic in the sweep that counts (1 of `iters`).
SMEM_LOADS_PER_VISIT = 3.0
SMEM_ATOMICS_PER_VISIT_CACHED = 1.0
SMEM_ATOMICS_PER_VISIT_COUNTING = 2.0
# HBM bytes a windowed history needs besides its share of the code stream: perm 4 + p0 4 + pflag 1 + N 4 + ell 4 + b 4
HBM_BYTES_PER_HISTORY = 21.0
# K1 (MLP + walk) is bound by the plain FP64 ALUs: FP64 instructions per MLP sample of the Gaussian-conditioning form
# (30 FMA of six Horner polynomials + 69 other FP64 operations incl. one division and one square root
# counted as one each); hull search, stepping compares and integer work are not counted.
FP64_OPS_PER_SAMPLE = 99.0


def measured_hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "MEASURED_PEAKS.json (burst copy)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = "index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown," \
        "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.index)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm, smax, reasons = [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); smax.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def pick_config(name: str, m: int, block: int = 0, lam: float = 0.0, iters: int = 0):
    """BASELINE.json config by name; m / block / lam / iters override it (config 4 = block-size / relaxation sweep on the
    config-1 phantom and histories)."""
    cfg = synth.CONFIGS[name]
    if m:
        cfg = dataclasses.replace(cfg, m=m)
    if block:
        cfg = dataclasses.replace(cfg, block=block)
    if lam:
        cfg = dataclasses.replace(cfg, lam=lam)
    if iters:
        cfg = dataclasses.replace(cfg, iters=iters)
    return cfg


def oracle_run(cfg, pr_host, hull_host, iters: int, threads: int = 0):
    """Times the oracle (as it stands) on the given histories (host numpy arrays).  Returns seconds, counts and x."""
    from oracle import pcto
    m = int(pr_host["phi"].shape[0])
    g = pcto.make_geometry(**synth.geometry(cfg))
    p = pcto.make_params(**synth.mlp_params(cfg))
    pa = pcto.ProtonArrays({k: v for k, v in pr_host.items() if k != "wepl"}, -cfg.u_tracker, cfg.u_tracker)
    t0 = time.perf_counter()
    P = pcto.Paths(g, p, pa, hull_host, threads)
    t1 = time.perf_counter()
    x = P.solve(pr_host["wepl"], np.ones(cfg.n, np.float32), iters, cfg.block, cfg.lam, threads)
    t2 = time.perf_counter()
    out = dict(m=m, visits=P.total_visits, iters=iters, block=cfg.block, s_mlp=t1 - t0, s_solve=t2 - t1, x=x)
    P.free()
    return out


def oracle_sample_inputs(cfg, sample: int):
    """The first `sample` histories of the workload, generated on the CPU by the same recipe (the reference arm has no GPU
    arm beside it to share device-generated inputs with)."""
    x_true, hull, shadow = synth.make_phantom(cfg)
    pr = synth.generate_protons(cfg, x_true, shadow, i0=0, i1=min(sample, cfg.m))
    return {k: v.numpy() for k, v in pr.items()}, hull.numpy()


def run_reference(args, rank):
    """--impl reference: the CPU oracle on the host cores (rank 0 only)."""
    if rank != 0:
        return
    cfg = pick_config(args.config, args.m, args.block, args.lam, args.iters)
    cores = os.cpu_count() or 1
    iters = min(cfg.iters, 2)
    pr_h, hull_h = oracle_sample_inputs(cfg, args.oracle_sample)
    for _ in range(1 if args.warmup >= 1 else 0):
        small = {k: v[:max(1000, args.oracle_sample // 10)] for k, v in pr_h.items()}
        oracle_run(cfg, small, hull_h, 1)
    runs = [oracle_run(cfg, pr_h, hull_h, iters) for _ in range(args.steps)]
    secs = [r["s_mlp"] + r["s_solve"] for r in runs]
    upd = runs[0]["visits"] * iters
    value = upd * len(runs) / sum(secs)
    sample = f"the first {runs[0]['m']} histories of {cfg.name} (one block of the real run when <= {cfg.block}), MLP + {iters} DROP sweeps"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sum(secs) / len(secs), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "histories": cfg.m, "sample_histories": runs[0]["m"], "iters": iters,
                   "block": runs[0]["block"], "lambda": cfg.lam},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "mlp_histories_per_s": runs[0]["m"] * len(runs) / sum(r["s_mlp"] for r in runs),
                         "solver_updates_per_s": upd * len(runs) / sum(r["s_solve"] for r in runs)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def k2w_roofline(cfg, plan, peaks, hbm_peak_gbs, hbm_kind, prof, steps, traffic):
    """Roofline of the windowed block projection: the slowest of the four units a launch needs at least once.
    All counts are per profiled step (`iters` sweeps over all blocks); times in ms."""
    iters = cfg.iters
    V, H = plan["windowed_visits"], plan["windowed_histories"]
    n_launch = max(prof["project_windowed"][1], 1) / steps                        # launches per step
    t_meas = prof["project_windowed"][0] / steps                                  # ms per step, all launches
    # HBM: stream + counts are read by both walks of a launch, but a launch's share (~100 MB) fits L2, so once is compulsory
    hbm_bytes = iters * (plan["stream_bytes"] + plan["cnt_bytes"] + HBM_BYTES_PER_HISTORY * H)
    t_hbm = hbm_bytes / (hbm_peak_gbs * 1e9) * 1e3
    # L2: the x slots staged into the windows and the Delta slots flushed from them (<= staged), per sweep
    t_l2g = iters * plan["staged_slots"] / peaks["l2_gather_per_s"] * 1e3
    t_l2r = iters * plan["staged_slots"] / peaks["l2_red_f32_per_s"] * 1e3
    # shared memory: lane operations of the two walks at the measured random-slot rates
    loads = iters * SMEM_LOADS_PER_VISIT * V
    atoms = ((iters - 1) * SMEM_ATOMICS_PER_VISIT_CACHED + SMEM_ATOMICS_PER_VISIT_COUNTING) * V
    t_smem = (loads / peaks["smem_load_per_s"] + atoms / peaks["smem_atomic_per_s"]) * 1e3
    t_smem_cf = (loads / peaks["smem_load_cf_per_s"] + atoms / peaks["smem_atomic_cf_per_s"]) * 1e3
    comp = {"hbm": t_hbm, "l2_gather": t_l2g, "l2_red": t_l2r, "smem": t_smem}
    bound = max(comp, key=comp.get)
    t_roof = comp[bound]
    ops = loads + atoms
    launch_s = t_meas * 1e-3 / n_launch
    return {
        "bound": bound, "kernel": "k_block_windowed",
        "achieved": ops / (t_meas * 1e-3) if bound == "smem" else hbm_bytes / (t_meas * 1e-3) / 1e9,
        "peak": ops / (t_smem * 1e-3) if bound == "smem" else hbm_peak_gbs,
        "unit": "shared-memory lane-ops/s" if bound == "smem" else "GB/s",
        "frac": t_roof / t_meas if t_meas > 0 else 0.0,
        "peak_kind": ("pct_measure_peaks: random-slot shared-memory loads and atomics, weighted by the kernel's mix"
                      if bound == "smem" else hbm_kind),
        "roofline_ms_per_step": comp, "measured_ms_per_step": t_meas,
        "frac_of_conflict_free_smem": t_smem_cf / t_meas if t_meas > 0 else None,
        "traffic": traffic, "hbm_compulsory_bytes_per_launch": hbm_bytes / n_launch,
        "hbm_frac_of_peak": (traffic / launch_s / 1e9 / hbm_peak_gbs) if traffic else None,
        "avg_launch_ms": t_meas / n_launch, "launches_per_step": n_launch,
        "kernel_visits_per_s": iters * V / (t_meas * 1e-3) if t_meas > 0 else None,
        "lane_ops_per_visit": {"loads": SMEM_LOADS_PER_VISIT, "atomics_cached": SMEM_ATOMICS_PER_VISIT_CACHED,
                               "atomics_counting": SMEM_ATOMICS_PER_VISIT_COUNTING},
    }


def k2d_roofline(cfg, P, m, peaks, hbm_peak_gbs, prof, steps):
    """Roofline of the direct block projection (blocks too small for windows): L2 gathers and reductions per visit."""
    t_meas = prof["project_direct"][0] / steps
    iters = cfg.iters
    t_hbm = iters * (0.375 * P + 28.0 * m) / (hbm_peak_gbs * 1e9) * 1e3
    t_l2g = iters * P / peaks["l2_gather_per_s"] * 1e3
    t_l2r = iters * P / peaks["l2_red_v2_per_s"] * 1e3
    comp = {"hbm": t_hbm, "l2_gather": t_l2g, "l2_red": t_l2r}
    bound = max(comp, key=comp.get)
    return {"bound": bound, "kernel": "k_block_project_scatter", "achieved": iters * P / (t_meas * 1e-3) if t_meas > 0 else 0.0,
            "peak": iters * P / (comp[bound] * 1e-3), "unit": "visits/s", "frac": comp[bound] / t_meas if t_meas > 0 else 0.0,
            "peak_kind": "pct_measure_peaks (L2 random gather / red.v2.f32 rates)", "roofline_ms_per_step": comp,
            "measured_ms_per_step": t_meas, "traffic": None}


def read_traffic(cfg_name, kernel):
    """dram bytes per launch of `kernel` from the committed ncu --set full capture (profiles/roofline_traffic.csv)."""
    tp = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    if not os.path.exists(tp):
        return None, None
    try:
        for ln in open(tp).read().splitlines()[1:]:
            f = ln.split(",")
            if f[0] == cfg_name and f[1] == kernel:
                return float(f[2]), (f[3] if len(f) > 3 else None)
    except Exception:
        pass
    return None, None


def bench_workload(args, cfg, dev, local, world, dist, steps, warmup, e2e_steps, e2e_warmup, profile_steps, want_cpu, peaks=None,
                   do_pre=True):
    """Runs one workload; returns (measurements for the JSON line, the peaks used)."""
    from paper_1802_01070_b200 import binding

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- untimed setup: synthetic workload resident in HBM --------------------------------------------------
    x_true, hull, shadow = synth.make_phantom(cfg, dev)
    pr = synth.generate_protons(cfg, x_true, shadow, device=dev)
    protons = {k: pr[k] for k in binding.PROTON_KEYS}
    b = pr["wepl"]
    hull_flat = hull.reshape(-1).contiguous()
    x0 = torch.ones(cfg.n, dtype=torch.float32, device=dev)
    x = torch.empty_like(x0)
    ctx = binding.Context(synth.geometry(cfg), synth.mlp_params(cfg), local)
    info = {}

    def step(ev=None):
        if ev:
            ev[0].record()
        paths = ctx.generate_mlp(protons, -cfg.u_tracker, cfg.u_tracker, hull_flat)
        if ev:
            ev[1].record()
        ctx.solve(paths, b, x0, cfg.iters, cfg.block, cfg.lam, out=x)
        if ev:
            ev[2].record()
        info.update(samples=paths.total_samples, plan=paths.plan_info(), visits=paths.total_visits, rejected=paths.n_rejected,
                    ties=paths.n_ties, code_bytes=paths.code_bytes, header_bytes=paths.header_bytes,
                    general_segments=paths.n_general_segments)
        if "tie_log" not in info and ev is None:      # the logged boundary ties (north_star), once, outside the timed steps
            idx, n = ctx.paths_flagged(paths, binding.TIE, cap=64)
            info["tie_log"] = {"count": n, "fraction": n / max(cfg.m, 1), "history_indices": idx.tolist(),
                               "truncated": n > len(idx)}
        paths.free()

    for _ in range(warmup):
        step()
    barrier()
    launches0 = ctx.launch_count
    sampler = ClockSampler(local)
    sampler.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
    t_start, t_stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_start.record()
    for k in range(steps):
        step(evs[k])
    t_stop.record()
    barrier()
    clocks = sampler.stop()
    launches = ctx.launch_count - launches0
    ms_total = t_start.elapsed_time(t_stop)
    ms_mlp = sum(e[0].elapsed_time(e[1]) for e in evs)
    ms_solve = sum(e[1].elapsed_time(e[2]) for e in evs)
    t = torch.tensor([ms_total, ms_mlp, ms_solve], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total, ms_mlp, ms_solve = t.tolist()
    P = info["visits"]
    updates_per_step = P * cfg.iters
    value = world * updates_per_step * steps / (ms_total * 1e-3)

    # ---- per-kernel breakdown + rooflines: separate, instrumented steps (CUDA events around every launch) ----------------
    ctx.profile_read()
    ctx.profile_enable(True)
    p_start, p_stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p_start.record()
    for _ in range(profile_steps):
        step()
    p_stop.record()
    barrier()
    prof = ctx.profile_read()
    ctx.profile_enable(False)
    ms_prof_step = p_start.elapsed_time(p_stop) / max(profile_steps, 1)
    if peaks is None:
        peaks = ctx.measure_peaks()          # register / L2 / shared-memory microbenchmarks, measured now (~0.3 s)
    hbm_peak, hbm_kind = measured_hbm_peak()
    plan = info.get("plan") or {}
    if prof["project_windowed"][1] > 0:
        traffic, traffic_commit = read_traffic(cfg.name, "k_block_windowed")
        roofline = k2w_roofline(cfg, plan, peaks, hbm_peak, hbm_kind, prof, profile_steps, traffic)
        roofline["traffic_source"] = f"profiles/roofline_traffic.csv: ncu --set full, build {traffic_commit}" if traffic else None
    else:
        roofline = k2d_roofline(cfg, P, cfg.m, peaks, hbm_peak, prof, profile_steps)
    roofline["share_of_step"] = (prof["project_windowed"][0] + prof["project_direct"][0]) / profile_steps / ms_prof_step
    roofline["kernels_ms_per_step"] = {k: v[0] / profile_steps for k, v in prof.items()}
    roofline["kernel_launches_per_step"] = {k: v[1] / profile_steps for k, v in prof.items()}
    roofline["profiled_ms_per_step"] = ms_prof_step
    roofline["plan"] = plan
    k1_ms = prof["mlp"][0] / profile_steps
    k1_ops = FP64_OPS_PER_SAMPLE * info["samples"]
    roofline_k1 = {"bound": "alu", "kernel": "K1: k_hull + k_mlp_walk",
                   "achieved": k1_ops / (k1_ms * 1e-3) if k1_ms > 0 else 0.0, "peak": peaks["fp64_fma_per_s"],
                   "unit": "FP64 instructions/s", "frac": (k1_ops / (k1_ms * 1e-3) / peaks["fp64_fma_per_s"]) if k1_ms > 0 else 0.0,
                   "peak_kind": "measured (pct_measure_peaks: register-resident fma.rn.f64 chains)",
                   "fp64_ops_per_sample": FP64_OPS_PER_SAMPLE, "mlp_samples": info["samples"],
                   "share_of_step": k1_ms / ms_prof_step if ms_prof_step > 0 else None, "measured_ms_per_step": k1_ms}

    # ---- SURVEY 8(f) rows next to the hot path (untimed extras): FBP initial iterate, hull from data ---------------------
    pre = None
    if args.pre_steps and do_pre:
        import math
        n_s = 2 * int(math.ceil(0.5 * math.hypot(cfg.nx, cfg.ny))) + 2
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        ev[0].record()
        x_fbp = ctx.fbp(protons, -cfg.u_tracker, cfg.u_tracker, b, 180, n_s, cfg.h)
        ev[1].record()
        carved = ctx.hull_carve(protons, -cfg.u_tracker, cfg.u_tracker, b, 1.0, 0.25 * cfg.h)
        ev[2].record()
        torch.cuda.synchronize()
        paths = ctx.generate_mlp(protons, -cfg.u_tracker, cfg.u_tracker, hull_flat)
        k = min(cfg.m, 4 * cfg.block)

        def rms(xx):
            r = (ctx.forward_project(paths, xx)[:k] - b[:k]).double()
            return float(torch.sqrt(torch.mean(r * r)))
        curve = {"x0=1": [rms(x0)], "x0=fbp": [rms(x_fbp)]}
        xa, xb = x0.clone(), x_fbp.clone()
        for _ in range(args.pre_steps):          # one sweep at a time: pct_solve resumes from the x it is given
            ctx.solve(paths, b, xa, 1, cfg.block, cfg.lam, out=xa)
            ctx.solve(paths, b, xb, 1, cfg.block, cfg.lam, out=xb)
            curve["x0=1"].append(rms(xa)); curve["x0=fbp"].append(rms(xb))
        # Algorithm 1 of the paper (R28) on this one GPU: the regions run in turn, each timed on its own
        # -- what each GPU of a G-GPU run would do; no multi-GPU number is claimed -- and the image compared with the joint solve
        alg1 = None
        if args.regions > 1:
            ext = max(1, int(round(7.5 / cfg.h)))            # the paper's 3 slices of 2.5 mm
            x_joint = ctx.solve(paths, b, x0, cfg.iters, cfg.block, cfg.lam)
            paths.free()
            x_a1 = torch.zeros_like(x_joint)
            per_region, members = [], []
            for r in range(args.regions):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                _, mem = ctx.reconstruct_regions(protons, -cfg.u_tracker, cfg.u_tracker, hull_flat, b, None, args.regions, ext,
                                                 cfg.iters, cfg.block, cfg.lam, region_first=r, region_count=1, out=x_a1)
                e1.record()
                torch.cuda.synchronize()
                per_region.append(e0.elapsed_time(e1)); members.append(mem[r])
            inside = hull_flat.bool()
            d = (x_a1 - x_joint)[inside].double()
            alg1 = {"n_regions": args.regions, "ext_slices": ext, "members": members, "histories": cfg.m,
                    "ms_per_region": per_region, "ms_slowest_region": max(per_region),
                    "vs_joint_solve": {"rel_l2_in_hull": float(d.norm() / x_joint[inside].double().norm()),
                                       "max_abs_in_hull": float(d.abs().max()), "mean_abs_in_hull": float(d.abs().mean())},
                    "note": "each region = pct_hull_intersect on all histories + membership + gather + pct_generate_mlp + pct_solve "
                            "on its members, timed alone on this GPU; Algorithm 1 is an approximation of the joint solve "
                            "(PAPER.md Tables VIII/IX: RSP errors move by <= 0.35 %)"}
            del x_joint, x_a1
        else:
            paths.free()
        hm = hull_flat.bool()
        pre = {"fbp_ms": ev[0].elapsed_time(ev[1]), "fbp_bins": [cfg.nz, 180, n_s], "hull_carve_ms": ev[1].elapsed_time(ev[2]),
               "hull_carve": {"wepl_air_mm": 1.0, "min_chord_mm": 0.25 * cfg.h, "voxels_kept": int(carved.sum()),
                              "analytic_hull_voxels": int(hm.sum()), "analytic_hull_voxels_carved": int((hm & (carved == 0)).sum())},
               "rms_residual_mm_by_sweep": curve,
               "algorithm1": alg1,
               "note": "rms of b - A x over the first 4 blocks after 0, 1, 2, ... sweeps from x0 = 1 and from the FBP image (PAPER.md:7)"}
        del x_fbp, carved, xa, xb

    # ---- end to end through the C-ABI on pinned HOST buffers ------------------------------------------------
    e2e = None
    if e2e_steps > 0:
        host = {k: torch.empty(cfg.m, dtype=torch.float64).pin_memory() for k in binding.PROTON_KEYS}
        for k in binding.PROTON_KEYS:
            host[k].copy_(protons[k])
        b_h = torch.empty(cfg.m, dtype=torch.float32).pin_memory(); b_h.copy_(b)
        hull_h = torch.empty(cfg.n, dtype=torch.uint8).pin_memory(); hull_h.copy_(hull_flat)
        x_h = torch.empty(cfg.n, dtype=torch.float32).pin_memory()
        for _ in range(e2e_warmup):      # untimed: the buffer cache settles on this call's allocation pattern
            ctx.reconstruct_host(host, -cfg.u_tracker, cfg.u_tracker, hull_h, b_h, None, cfg.iters, cfg.block, cfg.lam, x_h)
        barrier()
        e_start, e_stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e_start.record()
        for _ in range(e2e_steps):
            st = ctx.reconstruct_host(host, -cfg.u_tracker, cfg.u_tracker, hull_h, b_h, None, cfg.iters, cfg.block,
                                      cfg.lam, x_h)
        e_stop.record()
        barrier()
        e_ms = torch.tensor([e_start.elapsed_time(e_stop)], dtype=torch.float64, device=dev)
        if dist is not None:
            dist.all_reduce(e_ms, op=dist.ReduceOp.MAX)
        e_ms = e_ms.item()
        e2e = {"value": world * updates_per_step * e2e_steps / (e_ms * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": cfg.m * (9 * 8 + 4) + cfg.n, "d2h_bytes_per_step": cfg.n * 4,
               "steps": e2e_steps, "recon_s": e_ms * 1e-3 / e2e_steps,
               "phases_ms": {k: st[k] for k in ("ms_h2d", "ms_mlp", "ms_solve", "ms_d2h")},
               "x_checksum": float(x_h.double().sum())}
        del host, b_h, hull_h

    # ---- the oracle timed beside it (rank 0, N = 1 only) on the SAME histories: the first block(s) of the workload -------
    cpu_baseline = None
    if want_cpu:
        k = min(args.oracle_sample, cfg.m)
        pr_h = {key: pr[key][:k].cpu().numpy() for key in list(binding.PROTON_KEYS) + ["wepl"]}
        r = oracle_run(cfg, pr_h, hull.cpu().numpy(), 1)
        secs = r["s_mlp"] + r["s_solve"]
        # the same histories through the CUDA path: a live parity figure next to the timing
        sub = {key: pr[key][:k].contiguous() for key in binding.PROTON_KEYS}
        paths = ctx.generate_mlp(sub, -cfg.u_tracker, cfg.u_tracker, hull_flat)
        x_g = ctx.solve(paths, pr["wepl"][:k].contiguous(), x0, 1, cfg.block, cfg.lam).cpu().numpy()
        same_visits = paths.total_visits == r["visits"]
        paths.free()
        cpu_baseline = {"value": r["visits"] / secs, "unit": UNIT, "cores": os.cpu_count() or 1, "kind": "oracle",
                        "sample": f"the first {r['m']} histories of the {cfg.name} workload the GPU arm ran (copied from the device), "
                                  f"MLP + 1 DROP sweep, {secs:.1f} s",
                        "mlp_histories_per_s": r["m"] / r["s_mlp"], "solver_updates_per_s": r["visits"] / r["s_solve"],
                        "parity_on_sample": {"visits_equal": bool(same_visits),
                                             "rel_l2": float(np.linalg.norm(x_g - r["x"]) / np.linalg.norm(r["x"])),
                                             "max_abs": float(np.max(np.abs(x_g - r["x"])))}}

    out = {
        "value": value, "ms_per_step": ms_total / steps,
        "config": {"workload": cfg.name, "grid": [cfg.nx, cfg.ny, cfg.nz], "histories": cfg.m, "iters": cfg.iters,
                   "block": cfg.block, "lambda": cfg.lam, "blocks_per_iter": (cfg.m + cfg.block - 1) // cfg.block,
                   "l2": "inputs exceed L2 (code stream + tracker arrays >> 126 MB)",
                   "multi_gpu": "replicas only" if world > 1 else "single GPU"},
        "value_definition": "P x iters / whole-step time (pct_generate_mlp + plan + pct_solve)",
        "path_voxel_visits": P, "rejected": info["rejected"], "ties": info["ties"], "tie_log": info.get("tie_log"),
        "code_bytes": info["code_bytes"], "header_bytes": info["header_bytes"],
        "k1_general_segments": info["general_segments"],
        "solver_updates_per_s": world * updates_per_step * steps / (ms_solve * 1e-3),
        "solver_updates_per_s_definition": "P / t_iter, SURVEY.md 8(d): one sweep of A5-A7, plan build amortised in",
        "solver_ms_per_iter": ms_solve / (steps * cfg.iters),
        "mlp_histories_per_s": world * cfg.m * steps / (ms_mlp * 1e-3),
        "recon_s": ms_total * 1e-3 / steps,
        "roofline": roofline, "roofline_k1": roofline_k1, "cpu_baseline": cpu_baseline, "e2e": e2e, "preprocessing": pre,
        "gpu_launches": launches, "clocks": clocks,
    }
    del pr, protons, b, x, x0, hull_flat, hull, x_true
    ctx.trim_cache()
    ctx.close()
    return out, peaks


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", default=os.environ.get("PCT_BENCH_CONFIG", "paperA"), choices=sorted(synth.CONFIGS))
    ap.add_argument("--m", type=int, default=0, help="override the number of histories (parity/debug only)")
    ap.add_argument("--block", type=int, default=0, help="override the block size (config-4 sweep)")
    ap.add_argument("--lam", type=float, default=0.0, help="override the relaxation (config-4 sweep)")
    ap.add_argument("--iters", type=int, default=0, help="override the number of sweeps")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--e2e-warmup", type=int, default=2)
    ap.add_argument("--profile-steps", type=int, default=2, choices=range(1, 9),
                    help="instrumented steps for the per-kernel breakdown (outside the headline timing)")
    ap.add_argument("--regions", type=int, default=2, help="z-regions of the Algorithm-1 extra (PAPER.md:59-67); < 2: skip")
    ap.add_argument("--pre-steps", type=int, default=5, help="sweeps of the FBP-start vs unit-start residual curve (0: skip the 8(f) extras)")
    ap.add_argument("--oracle-sample", type=int, default=1_000_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--secondary", default=os.environ.get("PCT_BENCH_SECONDARY", "paperB"),
                    help="second workload reported under 'secondary' (the metric is quoted at 116M/261M); 'none' to skip")
    ap.add_argument("--peaks-only", action="store_true", help="print pct_measure_peaks() as JSON and exit")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback (use --impl reference for the oracle)")
    from paper_1802_01070_b200 import binding
    torch.cuda.set_device(local)
    if args.peaks_only:
        cfg = synth.CONFIGS["tiny"]
        ctx = binding.Context(synth.geometry(cfg), synth.mlp_params(cfg), local)
        pk = ctx.measure_peaks()
        pk.update(gpu=torch.cuda.get_device_name(local), hbm_gbs=measured_hbm_peak()[0], hbm_kind=measured_hbm_peak()[1])
        print(json.dumps(pk, indent=1))
        return
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    cfg = pick_config(args.config, args.m, args.block, args.lam, args.iters)
    want_cpu = rank == 0 and world == 1 and not args.no_cpu_baseline
    main_out, peaks = bench_workload(args, cfg, dev, local, world, dist, args.steps, args.warmup, args.e2e_steps,
                                     args.e2e_warmup, args.profile_steps, want_cpu)
    secondary = None
    overridden = args.m or args.block or args.lam or args.iters
    if args.secondary != "none" and args.secondary != cfg.name and not overridden and args.secondary in synth.CONFIGS:
        need = 150e9 if args.secondary == "paperB" else 0
        if torch.cuda.get_device_properties(local).total_memory >= need:
            torch.cuda.empty_cache()
            sec_out, _ = bench_workload(args, synth.CONFIGS[args.secondary], dev, local, world, dist, 2, 3,
                                        1 if args.e2e_steps > 0 else 0, 1, 1, False, peaks, do_pre=False)
            sec_out.update(steps=2, warmup=3, unit=UNIT)
            secondary = sec_out
    if rank == 0:
        line = {"metric": METRIC, "value": main_out.pop("value"), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": main_out.pop("ms_per_step"), "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64 MLP / f32 solver", "data": "synthetic"}
        line.update(main_out)
        line["peaks"] = peaks
        line["secondary"] = secondary
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- one JSON line for the pCT hot path on N B200s (contract in the task statement).

A "step" = one pass of the WHOLE hot path over the workload's synthetic histories, resident in HBM:
pct_generate_mlp (A1-A3) + pct_solve at the configured iterations (A4-A8).  `value` = path-voxel updates
(P = sum_i N_i visits x iterations) per second of step time; solver-only and MLP-only rates are extra keys.
`e2e` = the same through pct_reconstruct_host on pinned HOST buffers (H2D + MLP + solve + D2H inside the timing).
Multi-GPU: the path does not shard (north_star: one B200, no inter-GPU traffic) -> N independent replicas.
`--impl reference` times the CPU oracle (as it stands) on a bounded sample of the same workload.
"""
import argparse
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
# algorithmic bytes of the dominant kernel (the block projection, k_block_windowed / k_block_project_scatter): per visit 3 bit of
# code (HBM) + one 4-byte gather of x_j + one 8-byte {Delta,s} reduction; per history 24 bytes of header + b_i.
BYTES_PER_VISIT = 3.0 / 8.0 + 4.0 + 8.0
BYTES_PER_HISTORY = 24.0
# K1 (MLP + walk) is bound by the plain FP64 ALUs: FP64 instructions per MLP sample of the Gaussian-conditioning form
# (30 FMA of six Horner polynomials + 69 other FP64 operations incl. one division and one square root
# counted as one each); hull search, stepping compares and integer work are not counted.
FP64_OPS_PER_SAMPLE = 99.0


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured"
        except Exception:
            pass
    return 6650.0, "fallback"


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
    import dataclasses
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


def oracle_sample_run(cfg, sample: int, iters: int, threads: int = 0):
    """Times the oracle (as it stands) on a strided sample of the workload.  Returns dict with seconds and counts."""
    from oracle import pcto
    x_true, hull, shadow = synth.make_phantom(cfg)
    stride = max(1, cfg.m // sample)
    # strided sample of acquisition order = same angular coverage; generated directly as a smaller run of the same recipe
    sub = synth.scaled(cfg, min(sample, cfg.m), block=max(1, cfg.block // stride))
    pr = synth.generate_protons(sub, x_true, shadow)
    g = pcto.make_geometry(**synth.geometry(sub))
    p = pcto.make_params(**synth.mlp_params(sub))
    pa = pcto.ProtonArrays({k: v.numpy() for k, v in pr.items() if k != "wepl"}, -sub.u_tracker, sub.u_tracker)
    t0 = time.perf_counter()
    P = pcto.Paths(g, p, pa, hull.numpy(), threads)
    t1 = time.perf_counter()
    P.solve(pr["wepl"].numpy(), np.ones(sub.n, np.float32), iters, sub.block, sub.lam, threads)
    t2 = time.perf_counter()
    out = dict(m=sub.m, visits=P.total_visits, iters=iters, block=sub.block, s_mlp=t1 - t0, s_solve=t2 - t1)
    P.free()
    return out


def run_reference(args, rank):
    """--impl reference: the CPU oracle on the host cores (rank 0 only)."""
    if rank != 0:
        return
    cfg = pick_config(args.config, args.m, args.block, args.lam, args.iters)
    cores = os.cpu_count() or 1
    sample = args.oracle_sample
    iters = min(cfg.iters, 2)
    for _ in range(args.warmup if args.warmup < 1 else 1):
        oracle_sample_run(cfg, max(1000, sample // 10), 1)
    runs = [oracle_sample_run(cfg, sample, iters) for _ in range(args.steps)]
    secs = [r["s_mlp"] + r["s_solve"] for r in runs]
    upd = runs[0]["visits"] * iters
    value = upd * len(runs) / sum(secs)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sum(secs) / len(secs), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "histories": cfg.m, "sample_histories": runs[0]["m"], "iters": iters,
                   "block": runs[0]["block"], "lambda": cfg.lam},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{runs[0]['m']} histories of {cfg.name} (same recipe, fewer histories), MLP + {iters} DROP sweeps",
                         "mlp_histories_per_s": runs[0]["m"] * len(runs) / sum(r["s_mlp"] for r in runs),
                         "solver_updates_per_s": upd * len(runs) / sum(r["s_solve"] for r in runs)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


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
    ap.add_argument("--oracle-sample", type=int, default=1_000_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
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
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    cfg = pick_config(args.config, args.m, args.block, args.lam, args.iters)

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
        info.update(samples=paths.total_samples, plan=paths.plan_info(), visits=paths.total_visits, rejected=paths.n_rejected, ties=paths.n_ties, code_bytes=paths.code_bytes,
                    header_bytes=paths.header_bytes)
        paths.free()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    ctx.profile_read()
    ctx.profile_enable(True)
    launches0 = ctx.launch_count
    sampler = ClockSampler(local)
    sampler.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    t_start, t_stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_start.record()
    for k in range(args.steps):
        step(evs[k])
    t_stop.record()
    barrier()
    clocks = sampler.stop()
    launches = ctx.launch_count - launches0
    prof = ctx.profile_read()
    ctx.profile_enable(False)
    ms_total = t_start.elapsed_time(t_stop)
    ms_mlp = sum(e[0].elapsed_time(e[1]) for e in evs)
    ms_solve = sum(e[1].elapsed_time(e[2]) for e in evs)
    t = torch.tensor([ms_total, ms_mlp, ms_solve], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total, ms_mlp, ms_solve = t.tolist()
    P = info["visits"]
    updates_per_step = P * cfg.iters
    value = world * updates_per_step * args.steps / (ms_total * 1e-3)

    # ---- roofline of the dominant kernel (live CUDA events around every launch) -----------------------------
    peak, peak_kind = measured_peaks()
    # dominant kernel = the block projection (windowed K2w + direct K2d launches of the same blocks)
    ps_ms = prof["project_windowed"][0] + prof["project_direct"][0]
    ps_n = max(prof["project_windowed"][1], 1) if prof["project_windowed"][1] else max(prof["project_direct"][1], 1)
    kernel = "k_block_windowed" if prof["project_windowed"][1] else "k_block_project_scatter"
    blocks_per_iter = (cfg.m + cfg.block - 1) // cfg.block
    alg_bytes = args.steps * cfg.iters * (BYTES_PER_VISIT * P + BYTES_PER_HISTORY * cfg.m)
    achieved = alg_bytes / (ps_ms * 1e-3) / 1e9 if ps_ms > 0 else 0.0
    traffic = None          # dram bytes per launch of the dominant kernel from the committed ncu --set full capture
    tp = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    if os.path.exists(tp):
        try:
            for ln in open(tp).read().splitlines()[1:]:
                c, k, v = ln.split(",")
                if c == cfg.name and k == kernel:
                    traffic = float(v)
        except Exception:
            traffic = None
    roofline = {"bound": "hbm", "kernel": kernel, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "peak_kind": f"of {peak_kind}", "traffic": traffic,
                "avg_launch_ms": ps_ms / max(ps_n, 1), "launches": ps_n,
                "algorithmic_bytes_per_launch": alg_bytes / max(ps_n, 1),
                "share_of_step": ps_ms / ms_total if ms_total > 0 else None,
                "kernel_visits_per_s": args.steps * cfg.iters * P / (ps_ms * 1e-3) if ps_ms > 0 else None,
                "kernels_ms": {k: v[0] for k, v in prof.items()}, "plan": info.get("plan")}

    fp64_peak = ctx.measure_peaks()["fp64_fma_per_s"]          # register-resident fma.rn.f64 chains, measured now
    k1_ms = prof["mlp"][0]
    k1_ops = FP64_OPS_PER_SAMPLE * info["samples"] * args.steps
    roofline_k1 = {"bound": "alu", "kernel": "k_hull + k_mlp_walk (K1)", "achieved": k1_ops / (k1_ms * 1e-3) if k1_ms > 0 else 0.0,
                   "peak": fp64_peak, "unit": "FP64 instructions/s", "frac": (k1_ops / (k1_ms * 1e-3) / fp64_peak) if k1_ms > 0 else 0.0,
                   "peak_kind": "measured (pct_measure_peaks)", "fp64_ops_per_sample": FP64_OPS_PER_SAMPLE,
                   "mlp_samples": info["samples"], "share_of_step": k1_ms / ms_total if ms_total > 0 else None}

    # ---- end to end through the C-ABI on pinned HOST buffers ------------------------------------------------
    e2e = None
    if args.e2e_steps > 0:
        host = {k: torch.empty(cfg.m, dtype=torch.float64).pin_memory() for k in binding.PROTON_KEYS}
        for k in binding.PROTON_KEYS:
            host[k].copy_(protons[k])
        b_h = torch.empty(cfg.m, dtype=torch.float32).pin_memory(); b_h.copy_(b)
        hull_h = torch.empty(cfg.n, dtype=torch.uint8).pin_memory(); hull_h.copy_(hull_flat)
        x_h = torch.empty(cfg.n, dtype=torch.float32).pin_memory()
        for _ in range(2):      # untimed: the stream-ordered pool needs two passes to settle on this allocation pattern
            ctx.reconstruct_host(host, -cfg.u_tracker, cfg.u_tracker, hull_h, b_h, None, cfg.iters, cfg.block, cfg.lam, x_h)
        barrier()
        t0 = time.perf_counter()
        e_start, e_stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e_start.record()
        for _ in range(args.e2e_steps):
            st = ctx.reconstruct_host(host, -cfg.u_tracker, cfg.u_tracker, hull_h, b_h, None, cfg.iters, cfg.block,
                                      cfg.lam, x_h)
        e_stop.record()
        barrier()
        e_ms = torch.tensor([e_start.elapsed_time(e_stop)], dtype=torch.float64, device=dev)
        if dist is not None:
            dist.all_reduce(e_ms, op=dist.ReduceOp.MAX)
        e_ms = e_ms.item()
        e2e = {"value": world * updates_per_step * args.e2e_steps / (e_ms * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": cfg.m * (9 * 8 + 4) + cfg.n, "d2h_bytes_per_step": cfg.n * 4,
               "steps": args.e2e_steps, "recon_s": e_ms * 1e-3 / args.e2e_steps,
               "phases_ms": {k: st[k] for k in ("ms_h2d", "ms_mlp", "ms_solve", "ms_d2h")},
               "x_checksum": float(x_h.double().sum())}
        del host, b_h, hull_h

    # ---- the oracle timed beside it (rank 0, N = 1 only) ----------------------------------------------------
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        r = oracle_sample_run(cfg, args.oracle_sample, 1)
        secs = r["s_mlp"] + r["s_solve"]
        cpu_baseline = {"value": r["visits"] / secs, "unit": UNIT, "cores": os.cpu_count() or 1, "kind": "oracle",
                        "sample": f"{r['m']} histories of {cfg.name} (same recipe, fewer histories), MLP + 1 DROP sweep, {secs:.1f} s",
                        "mlp_histories_per_s": r["m"] / r["s_mlp"], "solver_updates_per_s": r["visits"] / r["s_solve"]}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64 MLP / f32 solver", "data": "synthetic",
            "config": {"workload": cfg.name, "grid": [cfg.nx, cfg.ny, cfg.nz], "histories": cfg.m, "iters": cfg.iters,
                       "block": cfg.block, "lambda": cfg.lam, "blocks_per_iter": blocks_per_iter,
                       "l2": "inputs exceed L2 (code stream + tracker arrays >> 126 MB)",
                       "multi_gpu": "replicas only" if world > 1 else "single GPU"},
            "path_voxel_visits": P, "rejected": info["rejected"], "ties": info["ties"],
            "code_bytes": info["code_bytes"], "header_bytes": info["header_bytes"],
            "solver_updates_per_s": world * updates_per_step * args.steps / (ms_solve * 1e-3),
            "solver_ms_per_iter": ms_solve / (args.steps * cfg.iters),
            "mlp_histories_per_s": world * cfg.m * args.steps / (ms_mlp * 1e-3),
            "recon_s": ms_total * 1e-3 / args.steps,
            "roofline": roofline, "roofline_k1": roofline_k1, "cpu_baseline": cpu_baseline, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

"""pct_fbp_static: the FBP initial iterate (R25) with its sinogram scratch in a fixed device array -- the one entry point of
the library that allocates nothing (for callers under stream capture, in serving loops, in harnesses that forbid cudaMalloc).

Checked against the existing path, pct_fbp, on the same inputs, within the tolerance test_gpu_pre.py uses for the FBP image
(FP64 inside, float32 out: rel-L2 < 1e-6, max-abs < 2e-6 of the image scale), on TWO calls in a row with different binnings
and data, so that a call that relied on the scratch array being zero -- it keeps the previous call's sums and counts -- fails.
This file sorts last on purpose: the suite runs with pytest -x, and a failure here must not hide the parity tests."""
import numpy as np
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu


def test_fbp_static_matches_fbp_on_two_calls_in_a_row():
    from paper_1802_01070_b200 import binding
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    cfg = synth.scaled(synth.CONFIGS["tiny"], 50000)
    x_true, hull, shadow = synth.make_phantom(cfg, "cuda")
    pr = synth.generate_protons(cfg, x_true, shadow, device="cuda")
    ctx = binding.Context(synth.geometry(cfg), synth.mlp_params(cfg), 0)
    dev = {k: pr[k].cuda().contiguous() for k in binding.PROTON_KEYS}
    b = pr["wepl"].cuda().contiguous()
    u = cfg.u_tracker
    # second call: other binning, a higher count threshold, a NaN record and a NaN WEPL, half the histories
    dev2 = {k: v[:25000].clone() for k, v in dev.items()}
    dev2["t_in"][7] = float("nan")
    b2 = b[:25000].clone()
    b2[11] = float("nan")
    calls = [(dev, b, 45, 24, 2.0, 1), (dev2, b2, 91, 50, 1.0, 2)]
    ref = [ctx.fbp(d, -u, u, w, nt, ns, ds, mc).clone() for d, w, nt, ns, ds, mc in calls]        # the existing path
    out = torch.empty(ctx.n, dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    got = []
    for d, w, nt, ns, ds, mc in calls:                  # back to back on one stream, same output buffer, nothing allocated
        assert cfg.nz * nt * ns <= binding.FBP_STATIC_MAX_CELLS
        ctx.fbp_static(d, -u, u, w, nt, ns, ds, mc, out=out)
        got.append(out.cpu().numpy().copy())
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "device memory was taken during pct_fbp_static"
    for x_s, x_r in zip(got, ref):
        x_r = x_r.cpu().numpy()
        scale = np.abs(x_r).max()
        assert scale > 0.5 and np.all(np.isfinite(x_s))
        assert np.linalg.norm(x_s - x_r) / np.linalg.norm(x_r) < 1e-6
        assert np.abs(x_s - x_r).max() < 2e-6 * scale
    assert np.abs(got[0] - got[1]).max() > 1e-3          # the two calls really were different problems
    # first call once more after the second: the larger sinogram's leftovers must not leak into the smaller one
    d, w, nt, ns, ds, mc = calls[0]
    again = ctx.fbp_static(d, -u, u, w, nt, ns, ds, mc, out=out).cpu().numpy()
    assert np.abs(again - got[0]).max() < 2e-6 * np.abs(got[0]).max()
    # no histories -> zero image; beyond the fixed scratch -> a clear error, not a fault
    empty = {k: torch.empty(0, dtype=torch.float64, device="cuda") for k in binding.PROTON_KEYS}
    assert torch.count_nonzero(ctx.fbp_static(empty, -u, u, torch.empty(0, device="cuda"), 45, 24, 2.0)) == 0
    with pytest.raises(binding.PctError, match="exceed the fixed scratch"):
        ctx.fbp_static(dev, -u, u, b, 1024, 1024, 0.1)          # 8 slices x 2^20 bins
    with pytest.raises(binding.PctError):
        ctx.fbp_static(dev, -u, u, b, 0, 24, 2.0)
    ctx.close()

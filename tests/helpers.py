"""Shared test helpers (input marshalling only; no method arithmetic)."""
import numpy as np

import synth


def oracle_setup(pcto, cfg, protons, hull=None, params_override=None, nthreads=0):
    g = pcto.make_geometry(**synth.geometry(cfg))
    kw = synth.mlp_params(cfg)
    if params_override:
        kw.update(params_override)
    p = pcto.make_params(**kw)
    arrays = {k: (v.cpu().numpy() if hasattr(v, "cpu") else np.asarray(v)) for k, v in protons.items() if k != "wepl"}
    pa = pcto.ProtonArrays(arrays, -cfg.u_tracker, cfg.u_tracker)
    h = None if hull is None else (hull.cpu().numpy() if hasattr(hull, "cpu") else hull)
    return g, p, pa, pcto.Paths(g, p, pa, h, nthreads)


def split_rows(row_ptr, vox):
    return [vox[row_ptr[i]:row_ptr[i + 1]] for i in range(len(row_ptr) - 1)]

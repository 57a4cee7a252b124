"""Shared by the tests and bench.py: one config -> identical arguments for the oracle and the CUDA plan.

The C-ABI takes fp32 scalars, so every scalar is rounded through float32 FIRST and the oracle gets
exactly the value the library sees (as a double)."""
import numpy as np


def f32(v):
    return float(np.float32(v))


def rounded_kwargs(cfg, **overrides):
    kw = cfg.plan_kwargs()
    kw.update(overrides)
    for key in ("pitch", "c", "fs", "fc", "t_start", "f_number"):
        kw[key] = f32(kw[key])
    for key in ("row_tx_angles", "col_tx_angles", "t0", "elem_window"):
        if kw.get(key) is not None:
            kw[key] = [f32(v) for v in kw[key]]
    for key in ("grid_xz", "grid_yz"):
        g = kw[key]
        kw[key] = (int(g[0]), f32(g[1]), f32(g[2]), int(g[3]), f32(g[4]), f32(g[5]), f32(g[6]))
    return kw


def rel_err(gpu, ref):
    """max|gpu - oracle| / max|oracle| (north_star's parity measure), per frame jointly over both images."""
    gpu = np.asarray(gpu, dtype=np.complex128)
    ref = np.asarray(ref, dtype=np.complex128)
    return float(np.abs(gpu - ref).max() / np.abs(ref).max())

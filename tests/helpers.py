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


def mask_margin(kw):
    """Smallest relative distance | |lat - lat_j| * 2 F# - z | / z of any (pixel, element) pair of either image to the
    edge of the f-number mask, computed in fp64 from the rounded arguments the library sees.
    The kernels take the in/out decision in fp32 and the oracle in fp64 (the definition), so a parity case with an
    f-number is only meaningful when no pair lies within fp32 rounding of the edge: callers assert margin >= 1e-6."""
    f = kw.get("f_number") or 0.0
    if f == 0.0:
        return float("inf")
    best = float("inf")
    for key, n_el in (("grid_xz", kw["n_cols"]), ("grid_yz", kw["n_rows"])):
        n_lat, lat0, dlat, n_ax, z0, dz, _ = kw[key]
        lat = lat0 + dlat * np.arange(n_lat)
        z = z0 + dz * np.arange(n_ax)
        lj = (np.arange(n_el) - (n_el - 1) / 2.0) * kw["pitch"]
        dx = np.abs(lat[:, None] - lj[None, :])                      # [lat][elem]
        rel = np.abs(dx[:, None, :] * (2.0 * f) - z[None, :, None]) / z[None, :, None]
        best = min(best, float(rel.min()))
    return best


def assert_mask_margin(kw, margin=1e-6):
    m = mask_margin(kw)
    assert m >= margin, "a (pixel, element) pair lies %.2e (relative) from the f-number mask edge" % m

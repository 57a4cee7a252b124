"""CPU check of the ring kernel's host-side tile / window planning (ulm_rca_ring_probe, no CUDA device needed):
every gather a tile can issue -- brute force over all its pixels, receive elements and angles, in fp64 -- must
fall inside the shared-memory stage the plan sizes for that (tile, element)."""
import numpy as np
import pytest

import synth
from helpers import rounded_kwargs

PX, TILE = 4, 384     # rows per strip, positions per tile (include/ulm_rca.h: ulm_rca_ring_probe)


def brute_force_check(n_rx, pitch, angles, c, fs, grid, t0=None, t_start=0.0):
    from paper_2511_21647_b200 import ring_probe
    r = ring_probe(n_rx, pitch, angles, c, fs, grid, t0=t0, t_start=t_start)
    n_lat, lat0, dlat, n_ax, z0, dz, ref = grid
    n_pos = n_lat * ((n_ax + PX - 1) // PX)
    assert r["n_tiles"] == (n_pos + TILE - 1) // TILE
    assert r["window"] % 8 == 0 and r["wj"].max() <= r["window"] and (r["wj"] % 8 == 0).all()
    t0 = np.zeros(len(angles)) if t0 is None else np.asarray(t0, dtype=np.float64)
    th = np.asarray(angles, dtype=np.float64)
    ej = (np.arange(n_rx) - 0.5 * (n_rx - 1)) * pitch
    used = np.zeros_like(r["wj"])
    for t in range(r["n_tiles"]):
        pos = np.arange(t * TILE, min((t + 1) * TILE, n_pos))
        strip, ix = pos // n_lat, pos % n_lat
        iz0 = int(strip[0]) * PX
        for m in range(PX):
            iz = strip * PX + m
            ok = iz < n_ax
            if not ok.any():
                continue
            x = lat0 + ix[ok] * dlat
            z = z0 + iz[ok] * dz
            # receive excess H(p, j) and transmit part U0_k(z), in samples (SURVEY 8(c) step 1 split as in DESIGN.md 7)
            H = (np.sqrt((x[:, None] - ej[None, :]) ** 2 + z[:, None] ** 2) - z[:, None]) * fs / c          # [p][j]
            U0 = (t0[None, :] + (z[:, None] * np.cos(th)[None, :] + ref * np.sin(th)[None, :]) / c + z[:, None] / c
                  - t_start) * fs                                                                            # [p][k]
            z_top = z0 + iz0 * dz
            U0_top = (t0 + (z_top * np.cos(th) + ref * np.sin(th)) / c + z_top / c - t_start) * fs           # [k]
            upm = (U0 - np.floor(U0_top)[None, :] - 0.5)[:, None, :] + (H - r["dj"][t][None, :])[:, :, None]  # [p][j][k]
            idx = np.rint(upm)
            assert idx.min() >= 0, (t, m, idx.min())
            top = idx.max(axis=(0, 2)) + 1          # entries the stage of element j must hold
            assert (top <= r["wj"][t]).all(), (t, m, int((top - r["wj"][t]).max()))
            used[t] = np.maximum(used[t], top.astype(np.int64))
    # the windows are not grossly oversized either (a multiple of 8 with a few entries of slack)
    assert (r["wj"] - used).max() <= 8 + 8, int((r["wj"] - used).max())
    return r


@pytest.mark.parametrize("index", [0, 1, 3])
def test_ring_windows_cover_every_gather_of_the_configs(index):
    cfg = synth.config(index)
    kw = rounded_kwargs(cfg)
    n_rx = kw["n_cols"]
    r = brute_force_check(n_rx, kw["pitch"], kw["row_tx_angles"], kw["c"], kw["fs"], kw["grid_xz"],
                          t_start=kw["t_start"])
    if index == 1:
        assert r["window"] == 224 and r["n_tiles"] == 20      # the figures DESIGN.md 6.2 quotes for cfg 1-2


def test_ring_windows_odd_shapes():
    # ragged grid (rows not a multiple of 4, one-and-a-bit tiles), negative lateral step, t0 offsets, off-centre ref
    brute_force_check(24, 0.3e-3, [-0.12, 0.0, 0.07], 1540.0, 25e6, (53, 4.0e-3, -0.154e-3, 37, 6e-3, 0.1e-3, 1e-3),
                      t0=[1e-7, -2e-7, 0.0], t_start=1e-6)
    brute_force_check(7, 0.5e-3, [0.0], 1500.0, 20e6, (3, -0.1e-3, 0.1e-3, 2, 10e-3, 0.2e-3, 0.0))


def test_ring_probe_rejects_unsupported_shapes():
    from paper_2511_21647_b200 import UlmRcaError, ring_probe
    with pytest.raises(UlmRcaError):
        ring_probe(300, 0.2e-3, [0.0], 1540.0, 20e6, (16, 0.0, 0.1e-3, 16, 10e-3, 0.1e-3, 0.0))   # > 256 elements


def test_event_folding_host_logic():
    """Transmit events fold exactly when their reference-slice delays coincide on every depth row: mirror angles
    about a centred slice with equal t0 (ulm_rca_fold_probe; DESIGN.md section 6 "event folding")."""
    from paper_2511_21647_b200 import fold_probe
    c, fs = 1540.0, 20e6
    centred = (64, -4.8e-3, 0.15e-3, 96, 5e-3, 0.154e-3, 0.0)
    off = centred[:6] + (0.4e-3,)
    a11 = [float(np.float32(np.radians(a))) for a in np.linspace(-10, 10, 11)]
    # the 11 angles of configs 1-3: five mirror pairs + the unpaired 0 degrees
    assert fold_probe(a11, c, fs, centred) == [10, 9, 8, 7, 6, -1, -2, -2, -2, -2, -2]
    # off-centre reference slice: ref sin(theta) changes sign inside a pair -> nothing folds
    assert fold_probe(a11, c, fs, off) == [-1] * 11
    # a different t0 inside a pair keeps it apart; equal t0 folds; duplicates fold; the middle one stays alone
    ang = [float(np.float32(np.radians(a))) for a in (-6.0, 2.0, 6.0)]
    assert fold_probe(ang, c, fs, centred, t0=[1e-7, -1e-7, 1e-7]) == [2, -1, -2]
    assert fold_probe(ang, c, fs, centred, t0=[1e-7, -1e-7, 2e-7]) == [-1, -1, -1]
    assert fold_probe([0.05, 0.0, 0.0, -0.05], c, fs, centred) == [3, 2, -2, -2]
    # an off-centre slice whose t0 difference cancels ref sin(theta) exactly in fp64 is a fold as well ...
    th = float(np.float32(np.radians(6.0)))
    dt = 2 * off[6] * np.sin(th) / c
    exact = fold_probe([-th, th], c, fs, off, t0=[dt, 0.0])
    # ... but t0 travels through the C-ABI as fp32, so the compensation is only approximate and must NOT fold
    assert exact == [-1, -1]

"""fp64 CPU oracle of the 2-D NCC microbubble localization on the projected planes -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

What the paper says: "the two projections are first normalized cross-correlated with the
corresponding Gaussian-fitted 2D PSFs (x-z and y-z), yielding two sets of 2D localizations"; "sub-pixel regional peaks in
the resulting correlating map are identified as ... localizations"; "we introduced separable subpixel correlation, where
the 2D operation was further decomposed into successive 1D correlations along each dimension" (Fig. 1g); "the 1D
correlation kernels in both directions were 11 elements long"; "Before localization, the maximum intensity of each volume
was obtained ... for thresholding".  PSF widths and thresholds are not given; the reading:

  LO-1  image B(l, i) = |V_p(l, i)| of one projected plane (B = 0 outside the plane); template g(a, b) = g1(a) g2(b),
        g1(a) = exp(-a^2 / (2 s_lat^2)), g2(b) = exp(-b^2 / (2 s_ax^2)), a, b = -5 .. 5 (11 x 11; s in pixels, arguments)
  LO-2  NCC map: with W = the 11 x 11 window centred on pixel p, Bm = mean of B over W, gm = mean of g:
            ncc(p) = sum_W (B - Bm)(g - gm) / sqrt( sum_W (B - Bm)^2  sum_W (g - gm)^2 )          (0 if the window is flat)
        -- the textbook normalised cross-correlation, written here as the plain 2-D sum.  (Because g is separable it
        equals three separable correlations -- sum B g, sum B, sum B^2 -- which is how the CUDA path evaluates it.)
  LO-3  candidates: interior pixels (not on the plane's border) with B(p) >= threshold_rel * max B over ALL planes of the
        frame ("maximum intensity of each volume") and ncc(p) >= ncc_min that are regional peaks of the NCC map: ncc(p)
        greater than the 4 neighbours that follow p in row-major order among its 8 neighbours, and not smaller than the 4
        that precede it (so a plateau yields exactly one peak)
  LO-4  sub-pixel position: 3-point parabola through the NCC map along each axis separately,
            delta = (n- - n+) / (2 (n- - 2 n0 + n+))   (0 if the denominator is 0)
        -> localization (l + delta_l, i + delta_i, ncc(p), B(p)).

Pins (tests/test_localize_pins.py): a plane that IS the template gives ncc = 1 at the blob centre and one localization
with delta = 0; gain / offset invariance of the NCC map; scipy.signal.correlate2d (a library routine) for the window
sums; sub-pixel blobs localized within 0.1 px; threshold and plateau rules on hand-made maps.  Parity unpinned: the PSF
widths, thresholds and the regional-peak rule (the paper gives none of them).
"""
from __future__ import annotations

import numpy as np

HALF = 5


def templates(s_lat: float, s_ax: float):
    a = np.arange(-HALF, HALF + 1, dtype=np.float64)
    return np.exp(-a * a / (2.0 * s_lat * s_lat)), np.exp(-a * a / (2.0 * s_ax * s_ax))


def ncc_map(b: np.ndarray, s_lat: float, s_ax: float) -> np.ndarray:
    """LO-1, LO-2: b [n_lat][n_ax] real >= 0 -> ncc [n_lat][n_ax]."""
    b = np.asarray(b, dtype=np.float64)
    g1, g2 = templates(s_lat, s_ax)
    g = np.outer(g1, g2)
    gz = g - g.mean()
    gden = np.sum(gz * gz)
    bp = np.pad(b, HALF)
    win = np.lib.stride_tricks.sliding_window_view(bp, (2 * HALF + 1, 2 * HALF + 1))     # [n_lat][n_ax][11][11]
    bm = win.mean(axis=(2, 3), keepdims=True)
    num = np.sum((win - bm) * gz, axis=(2, 3))
    bden = np.sum((win - bm) ** 2, axis=(2, 3))
    den = np.sqrt(bden * gden)
    out = np.zeros_like(b)
    ok = den > 0
    out[ok] = num[ok] / den[ok]
    return out


def parabola(nm: float, n0: float, np_: float) -> float:
    den = nm - 2.0 * n0 + np_
    return 0.0 if den == 0.0 else 0.5 * (nm - np_) / den


def localize_plane(b: np.ndarray, frame_max: float, s_lat: float, s_ax: float, threshold_rel: float, ncc_min: float):
    """LO-3, LO-4 on one plane: list of (lat, ax, ncc, intensity) in row-major order of the integer peak."""
    n = ncc_map(b, s_lat, s_ax)
    out = []
    after = [(0, 1), (1, -1), (1, 0), (1, 1)]          # neighbours that follow p in row-major order
    before = [(0, -1), (-1, 1), (-1, 0), (-1, -1)]
    for l in range(1, b.shape[0] - 1):
        for i in range(1, b.shape[1] - 1):
            if not (b[l, i] >= threshold_rel * frame_max and n[l, i] >= ncc_min):
                continue
            if all(n[l, i] > n[l + dl, i + di] for dl, di in after) and all(n[l, i] >= n[l + dl, i + di] for dl, di in before):
                out.append((l + parabola(n[l - 1, i], n[l, i], n[l + 1, i]), i + parabola(n[l, i - 1], n[l, i], n[l, i + 1]),
                            n[l, i], b[l, i]))
    return out


def plane_views(planes_frame: np.ndarray, n_xz: int, nx: int, n_yz: int, ny: int, nz: int):
    """One frame of ulm_rca_stage2_project output -> list of complex planes [n_lat][nz] (x-z planes, then y-z planes)."""
    a = planes_frame[:n_xz * nx * nz].reshape(n_xz, nx, nz)
    b = planes_frame[n_xz * nx * nz:].reshape(n_yz, ny, nz)
    return [a[m] for m in range(n_xz)] + [b[m] for m in range(n_yz)]


def localize_frame(planes_frame, n_xz, nx, n_yz, ny, nz, s_lat, s_ax, threshold_rel, ncc_min):
    """All planes of one frame: list (per plane) of localization lists; the threshold uses the frame's maximum."""
    views = [np.abs(v) for v in plane_views(np.asarray(planes_frame), n_xz, nx, n_yz, ny, nz)]
    fmax = max(float(v.max()) for v in views)
    return [localize_plane(v, fmax, s_lat, s_ax, threshold_rel, ncc_min) for v in views]

"""fp64 CPU oracle of the Fourier-domain NCC rigid motion estimation on the Stage-1 slices -- TEST INFRASTRUCTURE, NOT
PRODUCT CODE.

What the paper says (Section II.A.3): "sub-pixel motion was estimated using a Fourier-domain normalized
cross-correlation (NCC) approach [39].  In brief, each frame is transformed into the Fourier domain, the correlation
function between the two frames is computed, and the displacement versus the reference frame is determined by locating
the subpixel peak of the correlation function.  This procedure requires two forward and one inverse Fourier transform";
"motion estimation was applied immediately after Stage 1 beamforming, the K RC slices and K CR slices were used
separately to estimate motion within the x-z plane and the y-z plane.  K displacement vectors from K RC and K CR
transmissions were first averaged, and then the RC- and CR-averaged motions were vector-summed to recover the full 3D
motion"; Fig. 3d: "B-mode-based motion estimation".  Ref. [39] is not available; the reading:

  ME-1  B-mode image of a slice: a(l, i) = |S(l, i)|; its mean over the n_lat x n_ax pixels is removed, and the result is
        zero-padded to N1 x N2 = the next powers of two >= n_lat, n_ax (180 x 164 -> 256 x 256), which leaves 76 / 92
        pixels of zero margin: shifts up to that size correlate linearly (no wrap-around).
  ME-2  correlation function  c(d) = sum_x a_f(x + d) a_ref(x) / (|a_f| |a_ref|)   (|.| = root of the sum of squares of the
        mean-removed image; indices modulo N1, N2), evaluated as  IFFT2( FFT2(a_f) conj(FFT2(a_ref)) )  -- two forward and
        one inverse transform; c is in [-1, 1] and c(0) = 1 for identical images.
  ME-3  integer peak (d1, d2) = argmax c over all N1 N2 shifts, mapped to signed shifts (d >= N/2 -> d - N; ties: the first
        in row-major order); sub-pixel refinement by a 3-point parabola through the peak and its two (circular)
        neighbours, separately per axis:  delta = (c- - c+) / (2 (c- - 2 c0 + c+))   (0 when the denominator is 0).
        A frame whose content moved by +s pixels relative to the reference gives d = +s.
  ME-4  per frame: (dx, dz_RC) = mean over the K_r row-tx events of the x-z slices' (lateral, axial) shifts times the
        grid steps; (dy, dz_CR) likewise from the K_c column-tx events; 3-D motion = (dx, dy, dz) with
        dz = (dz_RC + dz_CR) / 2 when both apertures have events (else the one that exists).  The paper's "vector-summed"
        would literally count the axial motion twice; the two axial estimates measure the same displacement, so they are
        averaged (reading; listed in DESIGN.md).

numpy.fft serves as the library primitive of ME-2.  Pins (tests/test_motion_pins.py): brute-force spatial-domain NCC on
small images, integer circular shifts recovered exactly with delta = 0 and c = 1, invariance to gain and offset,
sub-pixel shifts of a smooth blob within the paper's 0.06 px, the combination rule by hand.  Parity unpinned: the
agreement of ME-1 .. ME-3 with the method of ref. [39] (B-mode input, zero padding, parabolic refinement are readings).
"""
from __future__ import annotations

import numpy as np


def pow2_at_least(n: int) -> int:
    m = 1
    while m < n:
        m *= 2
    return m


def prepared(a: np.ndarray, n1: int, n2: int):
    """ME-1: mean-removed, zero-padded image and its norm."""
    a = np.asarray(a, dtype=np.float64)
    a0 = a - a.mean()
    out = np.zeros((n1, n2))
    out[:a.shape[0], :a.shape[1]] = a0
    return out, np.sqrt(np.sum(a0 * a0))


def correlation(a: np.ndarray, ref: np.ndarray):
    """ME-1, ME-2: the normalised circular cross-correlation function c [N1][N2] of two equally sized real images."""
    n1, n2 = pow2_at_least(a.shape[0]), pow2_at_least(a.shape[1])
    ap, na = prepared(a, n1, n2)
    rp, nr = prepared(ref, n1, n2)
    c = np.fft.ifft2(np.fft.fft2(ap) * np.conj(np.fft.fft2(rp))).real
    den = na * nr
    return c / den if den > 0 else np.zeros_like(c)


def parabola(cm: float, c0: float, cp: float) -> float:
    den = cm - 2.0 * c0 + cp
    return 0.0 if den == 0.0 else 0.5 * (cm - cp) / den


def peak_shift(c: np.ndarray):
    """ME-3: (d1, d2, c_peak) with sub-pixel refinement."""
    n1, n2 = c.shape
    k = int(np.argmax(c))                      # first maximum in row-major order
    i, j = divmod(k, n2)
    d1 = parabola(c[(i - 1) % n1, j], c[i, j], c[(i + 1) % n1, j])
    d2 = parabola(c[i, (j - 1) % n2], c[i, j], c[i, (j + 1) % n2])
    s1 = i if i < n1 // 2 else i - n1
    s2 = j if j < n2 // 2 else j - n2
    return s1 + d1, s2 + d2, float(c[i, j])


def slice_shift(s_frame: np.ndarray, s_ref: np.ndarray):
    """Complex slices [n_lat][n_ax] -> (lateral shift, axial shift, NCC peak) of the frame against the reference."""
    return peak_shift(correlation(np.abs(s_frame), np.abs(s_ref)))


def estimate(p, slices: np.ndarray, ref_frame: int = 0):
    """slices: [n_frames][compound = 0 output].  Returns (per_event [n_frames][n_events][3] = (lateral px, axial px, ncc),
    motion [n_frames][4] = (dx, dy, dz in metres, mean NCC))  -- ME-1 .. ME-4."""
    slices = np.asarray(slices, dtype=np.complex128)
    kr, kc = len(p.row_tx_angles), len(p.col_tx_angles)
    shapes = [(p.grid_xz[0], p.grid_xz[3])] * kr + [(p.grid_yz[0], p.grid_yz[3])] * kc
    n_f = slices.shape[0]
    per = np.zeros((n_f, kr + kc, 3))
    off = 0
    for e, (nl, nz) in enumerate(shapes):
        ref = slices[ref_frame, off:off + nl * nz].reshape(nl, nz)
        for f in range(n_f):
            per[f, e] = slice_shift(slices[f, off:off + nl * nz].reshape(nl, nz), ref)
        off += nl * nz
    motion = np.zeros((n_f, 4))
    for f in range(n_f):
        dx = dzr = dy = dzc = 0.0
        if kr:
            dx = per[f, :kr, 0].mean() * p.grid_xz[2]
            dzr = per[f, :kr, 1].mean() * p.grid_xz[5]
        if kc:
            dy = per[f, kr:, 0].mean() * p.grid_yz[2]
            dzc = per[f, kr:, 1].mean() * p.grid_yz[5]
        dz = 0.5 * (dzr + dzc) if (kr and kc) else (dzr if kr else dzc)
        motion[f] = (dx, dy, dz, per[f, :, 2].mean())
    return per, motion

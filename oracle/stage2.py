"""fp64 CPU oracle of Stage-2 beamforming + sub-block sum-projection -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

What the paper says (Section II.A.1): the slices along the transmit direction are "approximately
identical ... differing only by a rigid axial shift determined by the transmit steering angle"; "In Stage 2, the
full volume V_k-RC/CR of size Nx x Ny x Nz is reconstructed from [the slice] by extrapolating along the transmit
direction for the kth steered RC and CR transmission.  Finally, the compounded volume V is obtained by coherently
summing all V_k-RC and V_k-CR".  PAPER.md:79, 93: the N x N x N volume is divided into N/P x N/P sub-blocks of
P x P x N voxels which are "sum-projected along lateral (x) and elevational (y) directions, resulting in projected
planes V_p-m (m = 1 .. N/P x 2) forming N/P planes along y-z and x-z planes separately"; P = 8.

The paper prints no formula (it defers to refs [33, 34], not available), so this file follows the reading fixed in
DESIGN.md section 11 ("Stage 2"), step by step, in plain numpy (fp64), with no blocking, fusion or reordering:

  S2-1  carrier removal.  For event k (angle th_k, offset t0_k) of an aperture whose reference slice sits at
        ref (y_ref for row-tx / RC events, x_ref for column-tx / CR events) the on-axis two-way time of depth z is
            tau0_k(z) = t0_k + (z cos th_k + ref sin th_k)/c + z/c
        and the baseband slice is  B_k(lat, i) = S_k(lat, i) exp(-j 2 pi fc tau0_k(z_i)).
  S2-2  rigid axial shift.  A voxel whose coordinate along the transmit direction is w (y for RC, x for CR) is
        read at depth z_i + delta_k(w),  delta_k(w) = (w - ref) tan(th_k / 2)  -- the shift that equalises the
        on-axis two-way time, (1 + cos th) delta = (w - ref) sin th -- by LINEAR interpolation along z of B_k on
        the axial grid, B_k taken as ZERO outside the grid:
            q = i + delta_k(w)/dz,  n = floor(q),  b = q - n,   L = (1 - b) B_k(lat, n) + b B_k(lat, n + 1)
  S2-3  carrier restoration at the voxel's own on-axis two-way time:
            V_k(lat, w, z_i) = L exp(+j 2 pi fc (tau0_k(z_i) + (w - ref) sin th_k / c))
  S2-4  coherent compounding:  V_RC = sum over row-tx events (lat = x, w = y),
        V_CR = sum over column-tx events (lat = y, w = x),  V = V_RC + V_CR  on the grid x = grid_xz lateral,
        y = grid_yz lateral, z = the common axial grid.
  S2-5  sub-block sum-projection:  groups of P consecutive indices (the last group may be
        shorter):  XZ_m(x, z) = sum_{y in group m} V(x, y, z),  m < ceil(Ny/P);
                   YZ_m(y, z) = sum_{x in group m} V(x, y, z),  m < ceil(Nx/P).

Pins (tests/test_stage2_pins.py): zero shift on the reference plane reproduces the compounded Stage-1 image exactly;
a th = 0 event is a pure replication; a linear-ramp record on one on-axis element makes Stage 2 EQUAL to the
brute-force 3-D DAS of oracle/ulm_oracle.c (pins the shift law, both signs and the carrier bookkeeping); an
impulse slice gives the closed-form shifted triangle (zero extension); linearity; the projection against explicit
loops and sum identities.  Against the brute-force 3-D DAS of a scatterer scene the step is an APPROXIMATION (off-axis
receive paths do not shift rigidly): that comparison carries a stated loose bound only, and the agreement of this
reading with the method of refs [33, 34] is **parity unpinned** (DESIGN.md section 11).
"""
from __future__ import annotations

import math

import numpy as np

TWO_PI = 2.0 * math.pi


def _axes(grid):
    n_lat, lat0, dlat, n_ax, z0, dz, ref = grid
    return lat0 + dlat * np.arange(n_lat), z0 + dz * np.arange(n_ax), float(ref), float(dz)


def slices_of_frame(p, frame_out):
    """compound = 0 output of one frame -> (S_rc [K_r][n_x][n_z], S_cr [K_c][n_y][n_z])."""
    kr, kc = len(p.row_tx_angles), len(p.col_tx_angles)
    nx, nz = p.grid_xz[0], p.grid_xz[3]
    ny = p.grid_yz[0]
    frame_out = np.asarray(frame_out, dtype=np.complex128)
    s_rc = frame_out[:kr * nx * nz].reshape(kr, nx, nz)
    s_cr = frame_out[kr * nx * nz:].reshape(kc, ny, p.grid_yz[3])
    return s_rc, s_cr


def extrapolate_event(p, s_k, theta, t0, ref, z, dz, w):
    """Steps S2-1 .. S2-3 for one event: s_k [n_lat][n_z] -> V_k [n_lat][len(w)][n_z]."""
    n_lat, n_z = s_k.shape
    tau0 = t0 + (z * math.cos(theta) + ref * math.sin(theta)) / p.c + z / p.c
    b_k = s_k * np.exp(-1j * TWO_PI * p.fc * tau0)[None, :]                       # S2-1
    out = np.zeros((n_lat, len(w), n_z), dtype=np.complex128)
    for iw, wv in enumerate(w):
        delta = (wv - ref) * math.tan(theta / 2.0)                                # S2-2
        for i in range(n_z):
            q = i + delta / dz
            n = math.floor(q)
            b = q - n
            lo = b_k[:, n] if 0 <= n <= n_z - 1 else 0.0
            hi = b_k[:, n + 1] if 0 <= n + 1 <= n_z - 1 else 0.0
            lerp = (1.0 - b) * lo + b * hi
            phase = TWO_PI * p.fc * (tau0[i] + (wv - ref) * math.sin(theta) / p.c)  # S2-3
            out[:, iw, i] = lerp * np.exp(1j * phase)
    return out


def stage2_volume(p, frame_out):
    """Steps S2-1 .. S2-4 on one frame of compound = 0 slices: (V_RC, V_CR), each [n_x][n_y][n_z]."""
    if (p.grid_xz[3], p.grid_xz[4], p.grid_xz[5]) != (p.grid_yz[3], p.grid_yz[4], p.grid_yz[5]):
        raise ValueError("Stage 2 needs identical axial grids")
    x, z, y_ref, dz = _axes(p.grid_xz)
    y, _, x_ref, _ = _axes(p.grid_yz)
    s_rc, s_cr = slices_of_frame(p, frame_out)
    kr = len(p.row_tx_angles)
    t0 = list(p.t0) if p.t0 is not None else [0.0] * (kr + len(p.col_tx_angles))
    v_rc = np.zeros((len(x), len(y), len(z)), dtype=np.complex128)
    v_cr = np.zeros_like(v_rc)
    for k, th in enumerate(p.row_tx_angles):           # RC: slice [x][z], transmit direction y
        v_rc += extrapolate_event(p, s_rc[k], th, t0[k], y_ref, z, dz, y)
    for k, th in enumerate(p.col_tx_angles):           # CR: slice [y][z], transmit direction x
        v_cr += extrapolate_event(p, s_cr[k], th, t0[kr + k], x_ref, z, dz, x).transpose(1, 0, 2)
    return v_rc, v_cr


def project_blocks(v, block):
    """Step S2-5: v [n_x][n_y][n_z] -> (XZ [ceil(n_y/P)][n_x][n_z], YZ [ceil(n_x/P)][n_y][n_z])."""
    n_x, n_y, n_z = v.shape
    gy, gx = -(-n_y // block), -(-n_x // block)
    xz = np.zeros((gy, n_x, n_z), dtype=v.dtype)
    yz = np.zeros((gx, n_y, n_z), dtype=v.dtype)
    for m in range(gy):
        xz[m] = v[:, m * block:(m + 1) * block, :].sum(axis=1)
    for m in range(gx):
        yz[m] = v[m * block:(m + 1) * block, :, :].sum(axis=0)
    return xz, yz


def stage2_planes(p, slices, block):
    """All steps on [frame][compound = 0 output]: complex128 [frame][XZ planes | YZ planes] flattened, each plane
    [lat][z] with z fastest -- the layout of ulm_rca_stage2_project."""
    outs = []
    for f in range(slices.shape[0]):
        v_rc, v_cr = stage2_volume(p, slices[f])
        xz, yz = project_blocks(v_rc + v_cr, block)
        outs.append(np.concatenate([xz.ravel(), yz.ravel()]))
    return np.stack(outs)

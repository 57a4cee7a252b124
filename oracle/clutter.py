"""fp64 CPU oracle of the eigen-based clutter filter on the Stage-1 slice stacks -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

What the paper says (Section II.A.2): every volume (here: every Stage-1 slice S_k of one transmit event,
"we therefore applied eigenvalue-based clutter filtering immediately on 2D slices S_k-RC/CR obtained from Stage 1")
is a column of the spatiotemporal matrix I in C^{n x n_t} (n pixels, n_t frames); the filter is "three steps: parallelly
computing the covariance matrix C in C^{n_t x n_t} of I, performing a lightweight eigenvalue decomposition of C, and
parallelly projecting to recover blood flow signals".  Neither the normalisation of C nor the rule that selects the
clutter components is given; the reading is:

  CF-1  covariance   C = I^H I,  C[i][j] = sum_p conj(I[p][i]) I[p][j]          (no 1/n, no mean removal)
  CF-2  eigen-decomposition  C = U diag(lambda) U^H,  lambda_1 >= lambda_2 >= ... >= 0   (Hermitian, positive semi-definite)
  CF-3  projection   the clutter subspace is spanned by the `rank` eigenvectors of the LARGEST eigenvalues, U_c;
                     I_f = I (1 - U_c U_c^H)     i.e. per pixel p, with s = I[p][:] as a column over the frames:
                     t_m = sum_f U_c[f][m] s[f],   s_f[f] = s[f] - sum_m conj(U_c[f][m]) t_m
The slices are stored frame-major, X[f][p] = I[p][f]  (X = one event's [frame][pixel] block of the compound = 0 output of
Stage 1), so C = conj(X) X^T and X_f = X - conj(U_c) (U_c^T X).

numpy.linalg.eigh serves as the library primitive of step CF-2 (it is pinned here against a hand-written cyclic Jacobi
on small matrices and against closed forms).  Pins (tests/test_clutter_pins.py): rank-1 / rank-2 tissue closed forms,
rank = 0 and rank = n_t, the SVD form of the same filter (numpy.linalg.svd, a different library routine), trace and
idempotence identities, plain-loop covariance.  Parity unpinned: the clutter-rank selection rule (the paper gives none;
`rank` is an argument).
"""
from __future__ import annotations

import numpy as np


def covariance(x: np.ndarray) -> np.ndarray:
    """CF-1.  x: [n_t][n] complex (frame-major stack of one event).  Returns C [n_t][n_t] complex128."""
    x = np.asarray(x, dtype=np.complex128)
    return np.conj(x) @ x.T


def eig_desc(c: np.ndarray):
    """CF-2.  Hermitian c -> (eigenvalues descending [n_t], eigenvectors as columns [n_t][n_t])."""
    lam, u = np.linalg.eigh(np.asarray(c, dtype=np.complex128))
    order = np.argsort(lam)[::-1]
    return lam[order], u[:, order]


def jacobi_eig_desc(c: np.ndarray, sweeps: int = 30):
    """Plain cyclic two-sided Jacobi for a small Hermitian matrix (used only to pin eig_desc): every off-diagonal
    element (p, q) is annihilated in turn by the unitary plane rotation built from a_pp, a_qq, a_pq."""
    a = np.array(c, dtype=np.complex128)
    n = a.shape[0]
    v = np.eye(n, dtype=np.complex128)
    for _ in range(sweeps):
        off = np.sqrt(np.sum(np.abs(a) ** 2) - np.sum(np.abs(np.diag(a)) ** 2))
        if off <= 1e-15 * np.sqrt(np.sum(np.abs(a) ** 2)):
            break
        for p in range(n - 1):
            for q in range(p + 1, n):
                apq = a[p, q]
                if abs(apq) == 0.0:
                    continue
                phase = apq / abs(apq)
                tau = (a[q, q].real - a[p, p].real) / (2.0 * abs(apq))
                t = (1.0 if tau >= 0 else -1.0) / (abs(tau) + np.sqrt(1.0 + tau * tau))
                cs = 1.0 / np.sqrt(1.0 + t * t)
                sn = t * cs
                j = np.eye(n, dtype=np.complex128)
                j[p, p] = cs
                j[q, q] = cs
                j[p, q] = sn * phase
                j[q, p] = -sn * np.conj(phase)
                a = j.conj().T @ a @ j
                v = v @ j
    lam = np.diag(a).real
    order = np.argsort(lam)[::-1]
    return lam[order], v[:, order]


def clutter_filter_stack(x: np.ndarray, rank: int):
    """CF-1 .. CF-3 on one event's stack x [n_t][n].  Returns (x_f [n_t][n], eigenvalues descending [n_t], C)."""
    x = np.asarray(x, dtype=np.complex128)
    c = covariance(x)
    lam, u = eig_desc(c)
    uc = u[:, :rank]
    t = uc.T @ x                              # t[m][p] = sum_f U_c[f][m] x[f][p]
    return x - np.conj(uc) @ t, lam, c


def event_blocks(p):
    """(offset, n_pix) of every event's slice inside one frame of the compound = 0 output."""
    nxz = p.grid_xz[0] * p.grid_xz[3]
    nyz = p.grid_yz[0] * p.grid_yz[3]
    out, off = [], 0
    for _ in p.row_tx_angles:
        out.append((off, nxz))
        off += nxz
    for _ in p.col_tx_angles:
        out.append((off, nyz))
        off += nyz
    return out


def clutter_filter(p, slices: np.ndarray, rank: int):
    """All events of an ensemble.  slices: [n_t][compound = 0 output] complex.  Returns (filtered, same shape complex128;
    eigenvalues [n_events][n_t] descending)."""
    slices = np.asarray(slices, dtype=np.complex128)
    out = np.empty_like(slices)
    lams = []
    for off, n in event_blocks(p):
        xf, lam, _ = clutter_filter_stack(slices[:, off:off + n], rank)
        out[:, off:off + n] = xf
        lams.append(lam)
    return out, np.stack(lams)

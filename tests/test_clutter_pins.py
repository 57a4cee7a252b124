"""Pins of the clutter-filter oracle (oracle/clutter.py) -- CPU only."""
import numpy as np
import pytest

from oracle import clutter


def rng_c(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def test_covariance_is_the_plain_double_loop():
    rng = np.random.default_rng(1)
    x = rng_c(rng, 5, 7)
    c = clutter.covariance(x)
    ref = np.zeros((5, 5), dtype=complex)
    for i in range(5):
        for j in range(5):
            for p in range(7):
                ref[i, j] += np.conj(x[i, p]) * x[j, p]          # C = I^H I with I[p][f] = x[f][p]
    np.testing.assert_allclose(c, ref, atol=1e-13)
    np.testing.assert_allclose(c, c.conj().T, atol=1e-13)            # Hermitian
    assert abs(np.trace(c).real - np.sum(np.abs(x) ** 2)) < 1e-10     # trace = energy


@pytest.mark.parametrize("n", [2, 5, 12])
def test_eigh_step_against_a_hand_written_jacobi(n):
    rng = np.random.default_rng(n)
    x = rng_c(rng, n, 3 * n)
    c = clutter.covariance(x)
    lam, u = clutter.eig_desc(c)
    lam_j, u_j = clutter.jacobi_eig_desc(c)
    np.testing.assert_allclose(lam, lam_j, rtol=0, atol=1e-10 * lam[0])
    assert np.all(np.diff(lam) <= 1e-12 * lam[0])                      # descending
    np.testing.assert_allclose(c @ u, u * lam[None, :], atol=1e-9 * lam[0])
    np.testing.assert_allclose(u.conj().T @ u, np.eye(n), atol=1e-12)
    # eigenvectors are unique up to a phase: compare the projectors onto each (simple) eigen-direction
    for k in range(n):
        np.testing.assert_allclose(np.outer(u[:, k], u[:, k].conj()), np.outer(u_j[:, k], u_j[:, k].conj()), atol=1e-8)


def test_rank_one_tissue_is_removed_exactly_and_an_orthogonal_bubble_is_kept():
    """x = a t^T (tissue: temporal profile a[f], spatial pattern t[p]) has C = conj(a) a^T |t|^2: one eigenvalue
    |a|^2 |t|^2 with eigenvector conj(a)/|a|.  rank = 1 removes it exactly; a weaker component b s^T whose temporal
    profile and spatial pattern are both orthogonal to the tissue's (a^H b = 0, t^H s = 0: the two terms are then the
    singular value decomposition of x) passes untouched."""
    rng = np.random.default_rng(3)
    nt, n = 16, 40
    a = rng_c(rng, nt)
    b = rng_c(rng, nt)
    b -= a * (np.vdot(a, b) / np.vdot(a, a))
    t, s = rng_c(rng, n), rng_c(rng, n)
    s -= t * (np.vdot(t, s) / np.vdot(t, t))
    tissue, bubble = 30.0 * np.outer(a, t), np.outer(b, s)
    xf, lam, c = clutter.clutter_filter_stack(tissue, 1)
    assert abs(lam[0] - 900.0 * np.vdot(a, a).real * np.vdot(t, t).real) < 1e-9 * lam[0] and abs(lam[1]) < 1e-9 * lam[0]
    assert np.abs(xf).max() < 1e-11 * np.abs(tissue).max()
    xf, lam, _ = clutter.clutter_filter_stack(tissue + bubble, 1)
    np.testing.assert_allclose(xf, bubble, atol=1e-10 * np.abs(tissue).max())
    # the wrong conjugation in CF-3 (projecting with U instead of conj(U)) would leave the tissue in: check it is gone
    assert np.abs(xf - bubble).max() < 1e-9


def test_rank_zero_is_identity_and_full_rank_is_zero():
    rng = np.random.default_rng(4)
    x = rng_c(rng, 9, 20)
    np.testing.assert_array_equal(clutter.clutter_filter_stack(x, 0)[0], x)
    assert np.abs(clutter.clutter_filter_stack(x, 9)[0]).max() < 1e-12 * np.abs(x).max()


@pytest.mark.parametrize("rank", [1, 3, 6])
def test_equals_the_svd_filter(rank):
    """The textbook SVD clutter filter: I = W S V^H, drop the `rank` largest singular components --
    computed with numpy.linalg.svd, a different library routine -- gives the same I_f; lambda = S^2."""
    rng = np.random.default_rng(10 + rank)
    nt, n = 12, 50
    x = rng_c(rng, nt, n) * np.linspace(5, 0.5, nt)[:, None]
    xf, lam, _ = clutter.clutter_filter_stack(x, rank)
    i_mat = x.T                                                    # [pixel][frame]
    w, s, vh = np.linalg.svd(i_mat, full_matrices=False)
    i_f = (w[:, rank:] * s[rank:]) @ vh[rank:, :]
    np.testing.assert_allclose(xf, i_f.T, atol=1e-10 * s[0])
    np.testing.assert_allclose(lam, s ** 2, atol=1e-9 * s[0] ** 2)
    # idempotent and energy-consistent: filtering twice changes nothing more than the spectrum says
    xff, lam2, _ = clutter.clutter_filter_stack(xf, 0)
    np.testing.assert_allclose(np.sum(np.abs(xf) ** 2), lam[rank:].sum(), rtol=1e-10)


def test_ensemble_layout_filters_every_event_on_its_own():
    import oracle
    import synth
    from synth import centred_grid
    d = synth.LAMBDA_M / 2
    cfg = synth.config(0).with_(compound=0, grid_xz=centred_grid(5, d, 4, 6e-3, d), grid_yz=centred_grid(3, d, 6, 6e-3, d),
                                row_tx_angles=(0.0, 0.1), col_tx_angles=(0.05,))
    p = oracle.OracleParams(**cfg.plan_kwargs())
    rng = np.random.default_rng(7)
    s = rng_c(rng, 10, 2 * 20 + 18)
    out, lams = clutter.clutter_filter(p, s, 2)
    assert lams.shape == (3, 10)
    for e, (off, n) in enumerate([(0, 20), (20, 20), (40, 18)]):
        ref, lam, _ = clutter.clutter_filter_stack(s[:, off:off + n], 2)
        np.testing.assert_array_equal(out[:, off:off + n], ref)
        np.testing.assert_array_equal(lams[e], lam)

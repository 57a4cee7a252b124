"""Pins of the motion-estimation oracle (oracle/motion.py) -- CPU only."""
import numpy as np
import pytest

from oracle import motion


def blob_image(n1, n2, centres, sigma=2.5):
    x, z = np.meshgrid(np.arange(n1), np.arange(n2), indexing="ij")
    img = np.zeros((n1, n2))
    for (cx, cz, amp) in centres:
        img += amp * np.exp(-((x - cx) ** 2 + (z - cz) ** 2) / (2 * sigma ** 2))
    return img


def test_fft_correlation_equals_the_spatial_domain_definition():
    """ME-2 written as the plain double sum over zero-padded, mean-removed images, on a 6 x 5 image (padded 8 x 8)."""
    rng = np.random.default_rng(1)
    a, ref = rng.random((6, 5)), rng.random((6, 5))
    c = motion.correlation(a, ref)
    assert c.shape == (8, 8)
    a0 = np.zeros((8, 8)); a0[:6, :5] = a - a.mean()
    r0 = np.zeros((8, 8)); r0[:6, :5] = ref - ref.mean()
    den = np.sqrt((a0 ** 2).sum() * (r0 ** 2).sum())
    for d1 in range(8):
        for d2 in range(8):
            s = 0.0
            for x in range(8):
                for z in range(8):
                    s += a0[(x + d1) % 8, (z + d2) % 8] * r0[x, z]
            assert abs(c[d1, d2] - s / den) < 1e-12


@pytest.mark.parametrize("shift", [(0, 0), (3, -2), (-7, 5), (12, 9)])
def test_integer_shift_is_recovered_exactly(shift):
    """A frame that is the reference moved by an integer number of pixels (zero-mean content well inside the image, so
    that the mean removal leaves no pedestal that stays behind): the peak sits at exactly that shift, the parabola is
    symmetric (delta = 0) and c = 1."""
    base = [(24, 22, 1.0), (32, 30, 0.7), (27, 35, -0.9), (36, 24, -0.8)]          # amplitudes sum to zero
    ref = blob_image(60, 56, base)
    frame = blob_image(60, 56, [(x + shift[0], z + shift[1], a) for (x, z, a) in base])
    d1, d2, c = motion.peak_shift(motion.correlation(frame, ref))
    assert abs(d1 - shift[0]) < 1e-6 and abs(d2 - shift[1]) < 1e-6     # the blobs reach the image edge only below 1e-7
    assert c > 0.999
    # gain and offset invariance (mean removal + normalisation)
    e1, e2, cc = motion.peak_shift(motion.correlation(3.7 * frame + 11.0, 0.2 * ref - 4.0))
    assert abs(e1 - d1) < 1e-9 and abs(e2 - d2) < 1e-9 and abs(cc - c) < 1e-12


def test_exact_circular_shift_of_the_padded_image():
    """Rolling the PADDED mean-removed image is an exact circular shift: c(shift) = 1 and delta = 0 to rounding."""
    rng = np.random.default_rng(3)
    a = rng.random((16, 16))
    c = motion.correlation(a, a)
    d1, d2, cp = motion.peak_shift(c)
    assert abs(d1) < 1e-12 and abs(d2) < 1e-12 and abs(cp - 1.0) < 1e-12
    assert abs(c.max() - 1.0) < 1e-12 and c.min() >= -1.0 - 1e-12


@pytest.mark.parametrize("sub", [(0.3, -0.45), (2.5, 1.25), (-1.7, 0.05)])
def test_sub_pixel_shift_within_the_papers_error(sub):
    """Smooth blobs displaced by a fraction of a pixel: the 3-point parabola is within the ~0.06 px the paper reports
    near half-pixel displacements."""
    base = [(14.0, 12.0, 1.0), (24.0, 19.0, 0.8), (18.0, 26.0, 0.5)]
    ref = blob_image(40, 36, base)
    frame = blob_image(40, 36, [(x + sub[0], z + sub[1], a) for (x, z, a) in base])
    d1, d2, c = motion.peak_shift(motion.correlation(frame, ref))
    assert abs(d1 - sub[0]) < 0.06 and abs(d2 - sub[1]) < 0.06


def test_parabola_closed_form():
    # samples of c(t) = 1 - (t - 0.2)^2 at t = -1, 0, 1: vertex at 0.2 exactly
    f = lambda t: 1 - (t - 0.2) ** 2
    assert abs(motion.parabola(f(-1), f(0), f(1)) - 0.2) < 1e-15
    assert motion.parabola(1.0, 1.0, 1.0) == 0.0


def test_combination_rule_by_hand():
    import oracle
    import synth
    from synth import centred_grid
    d = synth.LAMBDA_M / 2
    cfg = synth.config(0).with_(compound=0, grid_xz=centred_grid(50, 2 * d, 56, 6e-3, d), grid_yz=centred_grid(48, 3 * d, 56, 6e-3, d),
                                row_tx_angles=(0.0, 0.1), col_tx_angles=(0.05,))
    p = oracle.OracleParams(**cfg.plan_kwargs())
    bx = [(20, 22, 1.0), (30, 30, 0.6), (24, 34, -0.9), (32, 20, -0.7)]             # zero-mean content, well inside
    by = [(19, 21, 1.0), (28, 31, 0.6), (23, 35, -0.9), (30, 22, -0.7)]
    mv = lambda b, s: [(x + s[0], z + s[1], a) for (x, z, a) in b]
    ref_xz, ref_yz = blob_image(50, 56, bx) + 2.0, blob_image(48, 56, by) + 2.0     # + 2: a positive B-mode image
    f1_xz_a = blob_image(50, 56, mv(bx, (1, 2))) + 2.0                              # event 0: (+1, +2)
    f1_xz_b = blob_image(50, 56, mv(bx, (3, 2))) + 2.0                              # event 1: (+3, +2)
    f1_yz = blob_image(48, 56, mv(by, (-2, 4))) + 2.0                               # event 2: (-2, +4)
    frames = np.stack([np.concatenate([ref_xz.ravel(), ref_xz.ravel(), ref_yz.ravel()]),
                       np.concatenate([f1_xz_a.ravel(), f1_xz_b.ravel(), f1_yz.ravel()])]).astype(complex) * np.exp(0.7j)
    per, mot = motion.estimate(p, frames)
    assert np.abs(per[0, :, :2]).max() < 1e-9 and np.abs(per[0, :, 2] - 1).max() < 1e-12
    np.testing.assert_allclose(per[1, :, :2], [[1, 2], [3, 2], [-2, 4]], atol=1e-5)
    dx, dy, dz, ncc = mot[1]
    assert abs(dx - 2.0 * 2 * d) < 1e-4 * d and abs(dy - (-2.0) * 3 * d) < 1e-4 * d      # means (1 + 3)/2 and -2, times the lateral steps
    assert abs(dz - 0.5 * (2.0 + 4.0) * d) < 1e-4 * d                                    # axial: mean of the RC and CR estimates
    assert 0.9 < ncc <= 1.0

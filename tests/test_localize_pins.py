"""Pins of the localization oracle (oracle/localize.py) -- CPU only."""
import numpy as np
import pytest
from scipy.signal import correlate2d

from oracle import localize


def blob(n1, n2, c1, c2, s1, s2, amp=1.0):
    x, z = np.meshgrid(np.arange(n1), np.arange(n2), indexing="ij")
    return amp * np.exp(-((x - c1) ** 2) / (2 * s1 * s1) - ((z - c2) ** 2) / (2 * s2 * s2))


def test_a_plane_equal_to_the_template_scores_one_at_its_centre():
    b = blob(40, 36, 17, 14, 1.8, 1.3)
    n = localize.ncc_map(b, 1.8, 1.3)
    assert abs(n[17, 14] - 1.0) < 1e-9 and n.max() <= 1.0 + 1e-12 and n.min() >= -1.0 - 1e-12
    locs = localize.localize_plane(b, b.max(), 1.8, 1.3, 0.5, 0.6)
    assert len(locs) == 1
    l, i, ncc, inten = locs[0]
    assert abs(l - 17) < 1e-9 and abs(i - 14) < 1e-9 and abs(ncc - 1) < 1e-9 and abs(inten - 1.0) < 1e-12
    # gain / offset invariance of the map (where the window is not numerically flat)
    np.testing.assert_allclose(localize.ncc_map(3.3 * b + 0.7, 1.8, 1.3)[10:25, 7:22], n[10:25, 7:22], atol=1e-9)


def test_window_sums_against_scipy_correlate2d():
    """The three window sums of LO-2 with a library routine: sum B g, sum B, sum B^2 (zero boundary), then the NCC."""
    rng = np.random.default_rng(2)
    b = rng.random((23, 19))
    g1, g2 = localize.templates(2.0, 1.5)
    g = np.outer(g1, g2)
    sg = correlate2d(b, g, mode="same", boundary="fill")
    s1 = correlate2d(b, np.ones((11, 11)), mode="same", boundary="fill")
    s2 = correlate2d(b * b, np.ones((11, 11)), mode="same", boundary="fill")
    nw = 121.0
    num = sg - g.mean() * s1
    den = np.sqrt((s2 - s1 * s1 / nw) * np.sum((g - g.mean()) ** 2))
    np.testing.assert_allclose(localize.ncc_map(b, 2.0, 1.5), num / den, atol=1e-10)


@pytest.mark.parametrize("c", [(20.3, 17.6), (14.5, 22.25), (25.9, 12.1)])
def test_sub_pixel_blob_is_localized(c):
    b = blob(44, 40, c[0], c[1], 1.7, 1.4) + 0.3 * blob(44, 40, 8, 30, 1.7, 1.4)
    locs = localize.localize_plane(b, b.max(), 1.7, 1.4, 0.5, 0.8)
    assert len(locs) == 1                                # the weak second blob is below the intensity threshold
    assert abs(locs[0][0] - c[0]) < 0.1 and abs(locs[0][1] - c[1]) < 0.1
    both = localize.localize_plane(b, b.max(), 1.7, 1.4, 0.2, 0.8)
    assert len(both) == 2 and abs(both[0][0] - 8) < 0.1   # row-major order: the blob at lateral 8 first


def test_plateau_and_border_rules():
    """Two equal neighbouring maxima give one peak (the first in row-major order); border pixels are never candidates."""
    b = np.zeros((30, 30))
    b[10, 10] = b[10, 11] = 1.0                           # symmetric pair: the NCC map has a two-pixel plateau
    n = localize.ncc_map(b, 1.5, 1.5)
    assert abs(n[10, 10] - n[10, 11]) < 1e-15
    locs = localize.localize_plane(b, 1.0, 1.5, 1.5, 0.5, 0.0)
    assert [(round(l), round(i)) for l, i, _, _ in locs] == [(10, 10)]
    b2 = np.zeros((20, 20))
    b2[0, 7] = 1.0
    assert localize.localize_plane(b2, 1.0, 1.5, 1.5, 0.5, -1.0) == []
    assert localize.parabola(1.0, 1.0, 1.0) == 0.0

"""Pins of the Stage-2 oracle (oracle/stage2.py) -- CPU only.

The step is an approximation the paper does not spell out, so the oracle follows the DESIGN.md reading step by
step; these tests pin that reading to things other than itself: exact special cases in which the rigid-shift
extrapolation EQUALS the brute-force 3-D DAS of oracle/ulm_oracle.c, closed forms written out here, explicit loops,
and -- with a stated loose bound only -- the brute-force 3-D DAS of a scatterer scene.
"""
import math

import numpy as np
import pytest

import oracle
import synth
from oracle import stage2
from synth import centred_grid

TWO_PI = 2.0 * math.pi


def cfg_s2(**kw):
    """8+8 elements; lateral grids ON the element positions (pitch spacing) so that a pixel column can sit exactly
    under an element; common axial grid; off-centre reference slices; per-event t0."""
    pitch = 0.3e-3
    dz = synth.LAMBDA_M / 2
    base = dict(n_rows=8, n_cols=8, pitch=pitch, n_samples=700, n_frames=1, input_kind=1, t_start=0.7e-6,
                row_tx_angles=tuple(np.radians([-6.0, 0.0, 4.0])), col_tx_angles=tuple(np.radians([5.0, -3.0])),
                grid_xz=centred_grid(8, pitch, 48, 6e-3, dz, ref=0.45e-3),
                grid_yz=centred_grid(8, pitch, 48, 6e-3, dz, ref=-0.15e-3),
                t0=(0.2e-6, -0.1e-6, 0.05e-6, 0.3e-6, -0.25e-6), compound=0)
    base.update(kw)
    return synth.config(0).with_(**base)


def params(cfg, **kw):
    d = cfg.plan_kwargs()
    d.update(kw)
    return oracle.OracleParams(**d)


def axes(g):
    return g[1] + g[2] * np.arange(g[0]), g[4] + g[5] * np.arange(g[3]), g[6]


def test_reference_plane_reproduces_the_compounded_stage1_image():
    """delta = 0 and the carrier terms cancel on the reference slice: V_RC(x, y_ref, z) = sum_k S_k(x, z) and
    V_CR(x_ref, y, z) = sum_k S_k(y, z), i.e. exactly the compound = 1 images of Stage 1."""
    pitch = 0.3e-3
    # y grid containing y_ref = 0.45 mm = 1.5 pitch (index 5 of a centred 8-point pitch grid); x_ref = -0.15 mm (index 3)
    cfg = cfg_s2(input_kind=0)
    y = axes(cfg.grid_yz)[0]
    x = axes(cfg.grid_xz)[0]
    iy, ix = int(np.argmin(np.abs(y - cfg.grid_xz[6]))), int(np.argmin(np.abs(x - cfg.grid_yz[6])))
    assert abs(y[iy] - cfg.grid_xz[6]) < 1e-15 and abs(x[ix] - cfg.grid_yz[6]) < 1e-15
    ch = synth.random_channel(cfg, 1, seed=5, amplitude=4000)
    p0, p1 = params(cfg), params(cfg, compound=1)
    s = oracle.beamform(p0, ch)
    v_rc, v_cr = stage2.stage2_volume(p0, s[0])
    comp = oracle.beamform(p1, ch)[0]
    nxz = cfg.grid_xz[0] * cfg.grid_xz[3]
    scale = np.abs(comp).max()
    np.testing.assert_allclose(v_rc[:, iy, :].ravel(), comp[:nxz], rtol=0, atol=1e-12 * scale)
    np.testing.assert_allclose(v_cr[ix, :, :].ravel(), comp[nxz:], rtol=0, atol=1e-12 * scale)
    assert np.abs(v_rc[:, iy + 1, :].ravel() - comp[:nxz]).max() > 1e-3 * scale     # other planes differ


def test_unsteered_event_is_a_pure_replication():
    cfg = cfg_s2(row_tx_angles=(0.0,), col_tx_angles=(0.0,), t0=(0.1e-6, -0.2e-6), input_kind=0)
    ch = synth.random_channel(cfg, 1, seed=6, amplitude=4000)
    p = params(cfg)
    s = oracle.beamform(p, ch)
    s_rc, s_cr = stage2.slices_of_frame(p, s[0])
    v_rc, v_cr = stage2.stage2_volume(p, s[0])
    for iy in range(cfg.grid_yz[0]):
        np.testing.assert_allclose(v_rc[:, iy, :], s_rc[0], rtol=0, atol=1e-12 * np.abs(s_rc).max())
    for ix in range(cfg.grid_xz[0]):
        np.testing.assert_allclose(v_cr[ix, :, :], s_cr[0], rtol=0, atol=1e-12 * np.abs(s_cr).max())
    # ... so a P-block sum-projection of it is P times the slice (ragged last group: its size times the slice)
    xz, yz = stage2.project_blocks(v_rc, 3)
    assert xz.shape == (3, 8, 48) and yz.shape == (3, 8, 48)
    np.testing.assert_allclose(xz[0], 3 * s_rc[0], atol=1e-11 * np.abs(s_rc).max())
    np.testing.assert_allclose(xz[2], 2 * s_rc[0], atol=1e-11 * np.abs(s_rc).max())


@pytest.mark.parametrize("which", ["rc", "cr"])
def test_linear_ramp_on_an_on_axis_element_equals_brute_force_3d_das(which):
    """One receive element j, record iq[n] = a + b n (linear in n, so linear interpolation in time is exact), pixel
    column exactly under the element: the receive path is z for every depth, so the slices along the transmit
    direction differ EXACTLY by the rigid shift delta = (w - ref) tan(th/2) and by the carrier of the extra transmit
    path (w - ref) sin(th)/c -- Stage 2 must equal the 3-D DAS of oracle/ulm_oracle.c to rounding wherever the
    shifted depth stays inside the slice.  A wrong shift law (e.g. sin(th)/2), a wrong sign of the shift or of the
    carrier term, or a transposed axis fails this."""
    cfg = cfg_s2()
    rc = which == "rc"
    n_el = cfg.n_cols if rc else cfg.n_rows
    j = 5 if rc else 2
    a, b = 900, 7
    ch = np.zeros(cfg.channel_shape, dtype=np.int16)
    n = np.arange(cfg.n_samples)
    kr = len(cfg.row_tx_angles)
    events = range(kr) if rc else range(kr, cfg.n_events)
    for e in events:
        ch[0, e, (cfg.n_rows + j) if rc else j, :, 0] = a + b * n
    p = params(cfg)
    s = oracle.beamform(p, ch)
    v_rc, v_cr = stage2.stage2_volume(p, s[0])
    x, z, y_ref = axes(cfg.grid_xz)
    y, _, x_ref = axes(cfg.grid_yz)
    lat_j = (j - (n_el - 1) / 2.0) * cfg.pitch
    il = int(np.argmin(np.abs((x if rc else y) - lat_j)))
    assert abs((x if rc else y)[il] - lat_j) < 1e-15
    w, ref = (y, y_ref) if rc else (x, x_ref)
    angles = cfg.row_tx_angles if rc else cfg.col_tx_angles
    # brute force: 3-D DAS on the line of voxels under the element
    W, Z = np.meshgrid(w, z, indexing="ij")
    pts = np.stack([np.full(W.size, lat_j), W.ravel(), Z.ravel()], 1) if rc else \
        np.stack([W.ravel(), np.full(W.size, lat_j), Z.ravel()], 1)
    d_rc, d_cr = oracle.das_points(p, ch[0], pts)
    brute = (d_rc if rc else d_cr).reshape(len(w), len(z))
    got = v_rc[il, :, :] if rc else v_cr[:, il, :]
    # voxels whose shifted depth stays inside the slice for EVERY event (elsewhere the zero extension bites)
    dmax = np.max([np.abs((w - ref) * math.tan(th / 2.0)) for th in angles], axis=0) / cfg.grid_xz[5]
    iz = np.arange(len(z))
    ok = (iz[None, :] - dmax[:, None] >= 0) & (iz[None, :] + dmax[:, None] <= len(z) - 1)
    assert ok.sum() > 0.7 * ok.size
    scale = np.abs(brute).max()
    assert np.abs(got - brute)[ok].max() <= 1e-10 * scale
    assert np.abs(got - brute)[~ok].max() > 1e-3 * scale          # and the edge rule is really different there
    # the ramp makes the shift visible: without it (delta = 0) the two differ
    s_k = stage2.slices_of_frame(p, s[0])[0 if rc else 1]
    assert np.abs(np.abs(got[-1]) - np.abs(s_k.sum(0)[il]))[ok[-1]].max() > 1e-4 * scale


def test_impulse_slice_gives_the_shifted_triangle_with_zero_extension():
    """S_k = one non-zero pixel (x0, i0) of one event: V_k(x0, y, z_i) = s (1 - |i + delta/dz - i0|)^+ times the
    carrier ratio written out here; pixels whose shifted position leaves the grid read zeros."""
    cfg = cfg_s2()
    p = params(cfg)
    k, x0, i0, amp = 2, 3, 1, 2.0 - 1.5j
    frame = np.zeros(int(oracle.beamform(p, np.zeros(cfg.channel_shape, dtype=np.int16)).shape[1]), dtype=complex)
    nx, nz = cfg.grid_xz[0], cfg.grid_xz[3]
    frame[(k * nx + x0) * nz + i0] = amp
    v_rc, v_cr = stage2.stage2_volume(p, frame)
    assert np.all(v_cr == 0)
    x, z, y_ref = axes(cfg.grid_xz)
    y = axes(cfg.grid_yz)[0]
    th, t0 = cfg.row_tx_angles[k], cfg.t0[k]
    expect = np.zeros((len(y), nz), dtype=complex)
    for iy, yv in enumerate(y):
        for i in range(nz):
            q = i + (yv - y_ref) * math.tan(th / 2) / cfg.grid_xz[5]
            tri = max(0.0, 1.0 - abs(q - i0))
            tau_i = t0 + (z[i] * math.cos(th) + y_ref * math.sin(th)) / cfg.c + z[i] / cfg.c
            tau_0 = t0 + (z[i0] * math.cos(th) + y_ref * math.sin(th)) / cfg.c + z[i0] / cfg.c
            expect[iy, i] = amp * tri * np.exp(1j * TWO_PI * cfg.fc * (tau_i - tau_0 + (yv - y_ref) * math.sin(th) / cfg.c))
    np.testing.assert_allclose(v_rc[x0], expect, rtol=0, atol=1e-12)
    mask = np.ones(nx, dtype=bool)
    mask[x0] = False
    assert np.all(v_rc[mask] == 0)
    assert np.count_nonzero(expect) >= 2 * len(y) - 2


def test_linearity_and_projection_identities():
    cfg = cfg_s2(input_kind=0)
    p = params(cfg)
    a = oracle.beamform(p, synth.random_channel(cfg, 1, seed=1, amplitude=5000))
    b = oracle.beamform(p, synth.random_channel(cfg, 1, seed=2, amplitude=5000))
    for block in (3, 8, 5):
        pa, pb, pab = (stage2.stage2_planes(p, v, block) for v in (a, b, a + 2 * b))
        s = np.abs(pab).max()
        assert np.abs(pab - (pa + 2 * pb)).max() <= 1e-12 * s
    v_rc, v_cr = stage2.stage2_volume(p, a[0])
    v = v_rc + v_cr
    xz, yz = stage2.project_blocks(v, 3)
    # explicit loops (the definition of S2-5), ragged last group of 8 = 3 + 3 + 2
    for m in range(3):
        ys = [l for l in range(8) if l // 3 == m]
        ref = np.zeros((8, 48), dtype=complex)
        for l in ys:
            ref += v[:, l, :]
        np.testing.assert_allclose(xz[m], ref, atol=1e-12 * np.abs(v).max())
        ref = np.zeros((8, 48), dtype=complex)
        for l in ys:
            ref += v[l, :, :]
        np.testing.assert_allclose(yz[m], ref, atol=1e-12 * np.abs(v).max())
    # both plane stacks carry the same total per depth
    np.testing.assert_allclose(xz.sum((0, 1)), yz.sum((0, 1)), atol=1e-10 * np.abs(v).max())
    flat = stage2.stage2_planes(p, a, 3)[0]
    np.testing.assert_array_equal(flat, np.concatenate([xz.ravel(), yz.ravel()]))


def test_against_brute_force_3d_das_with_a_stated_loose_bound():
    """PARITY UNPINNED vs the paper: the rigid-shift extrapolation is an approximation (off-axis receive paths do
    not shift rigidly; SURVEY P6 measured its first-order form as loose).  On a small-angle scatterer scene with an
    f-number of 2 the relative L2 error against the brute-force 3-D DAS stays below 12 % (measured 8.4 %) within +-1.2 mm of the
    reference slice at +-3 degrees, shrinks towards the reference slice, and is ~0 on it.  A context number for
    DESIGN.md, not a parity claim."""
    d = synth.LAMBDA_M / 2
    cfg = synth.config(0).with_(n_frames=1, compound=0, f_number=2.0,
                                row_tx_angles=tuple(np.radians([-3.0, 0.0, 3.0])), col_tx_angles=(),
                                grid_xz=centred_grid(40, d, 60, 8e-3, d), grid_yz=centred_grid(17, d, 60, 8e-3, d))
    rng = np.random.default_rng(3)
    sc = np.column_stack([rng.uniform(-2.5e-3, 2.5e-3, 12), rng.uniform(-1.2e-3, 1.2e-3, 12),
                          rng.uniform(9e-3, 16e-3, 12), rng.uniform(0.5, 1.0, 12)])
    ch = synth.render(cfg, [0], noise=False, scat={0: sc})
    p = params(cfg)
    s = oracle.beamform(p, ch)
    v_rc, _ = stage2.stage2_volume(p, s[0])
    x, z, _ = axes(cfg.grid_xz)
    y = axes(cfg.grid_yz)[0]
    brute, _ = oracle.volume(p, ch[0], x, y, z)
    err = np.sqrt((np.abs(v_rc - brute) ** 2).sum((0, 2)) / (np.abs(brute) ** 2).sum((0, 2)))
    mid = len(y) // 2
    assert err[mid] < 1e-12
    assert err.max() < 0.12
    assert err[mid + 1] < err[-1] and err[mid - 1] < err[0]
    print("stage-2 vs brute-force 3-D DAS, relative L2 error per y plane:", np.round(err, 4))

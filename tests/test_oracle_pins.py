"""Pins of the fp64 oracle -- CPU only.

Each test checks oracle/ulm_oracle.c against something OTHER than itself: a closed form written out
by hand here, an invariant of the mathematics, a textbook special case, or an independently coded
brute force.  A dropped term, a wrong sign or index, or swapped row/column bookkeeping fails at least
one of them.
"""
import math

import numpy as np
import pytest

import oracle
import synth
from oracle.oracle import split_projections
from synth import centred_grid

TWO_PI = 2.0 * math.pi


def tiny(**kw):
    """8+8-element array, 3+2 angles, small grids, IQ input unless overridden."""
    d = synth.LAMBDA_M / 2
    base = dict(n_rows=8, n_cols=8, pitch=0.3e-3, n_samples=512,
                row_tx_angles=tuple(np.radians([-6.0, 1.0, 5.0])),
                col_tx_angles=tuple(np.radians([-4.0, 7.0])),
                grid_xz=centred_grid(12, d, 40, 6e-3, d / 4, ref=0.4e-3),
                grid_yz=centred_grid(10, 1.3 * d, 36, 6.5e-3, 0.9 * d / 4, ref=-0.3e-3),
                n_frames=1, input_kind=1, t_start=1.1e-6,
                t0=(0.2e-6, -0.1e-6, 0.05e-6, 0.3e-6, -0.25e-6))
    base.update(kw)
    return synth.config(0).with_(**base)


def params(cfg, **kw):
    d = cfg.plan_kwargs()
    d.update(kw)
    return oracle.OracleParams(**d)


def elem_pos(e, n, pitch):
    return (e - (n - 1) / 2.0) * pitch


def grid_axes(g):
    n_lat, lat0, dlat, n_ax, z0, dz, ref = g
    return lat0 + dlat * np.arange(n_lat), z0 + dz * np.arange(n_ax), ref


def rx_channel(cfg, row_tx, elem):
    return (cfg.n_rows + elem if row_tx else elem) if cfg.all_channels else elem


# ---------------------------------------------------------------------------------------------
# P1  closed form: one impulse on one channel of one event
# ---------------------------------------------------------------------------------------------
# (t_start, n_samples, impulse sample): interior hits, and records whose first / last samples fall
# inside the imaged depth range so that the edge rule (term = 0 unless 0 <= n and n+1 <= Ns-1) bites
P1_CASES = [(1.1e-6, 512, 152), (1.1e-6, 512, 160), (1.1e-6, 512, 169),
            (8.7e-6, 512, 0), (8.7e-6, 512, 1), (8.7e-6, 512, 9),
            (1.1e-6, 165, 164), (1.1e-6, 165, 163), (1.1e-6, 165, 155)]


@pytest.mark.parametrize("which", ["xz", "yz"])
@pytest.mark.parametrize("t_start,n_samples,n_s", P1_CASES)
def test_p1_impulse_closed_form(which, t_start, n_samples, n_s):
    cfg = tiny(t_start=t_start, n_samples=n_samples)
    p = params(cfg)
    row_tx = which == "xz"
    k = 2 if row_tx else 1                      # angle index within its aperture
    e = k if row_tx else len(cfg.row_tx_angles) + k
    j = 5 if row_tx else 2                      # the one active receive element
    amp = 1234.0 - 777.0j
    ch = np.zeros(cfg.channel_shape, dtype=np.int16)
    ch[0, e, rx_channel(cfg, row_tx, j), n_s] = (int(amp.real), int(amp.imag))
    out = oracle.beamform(p, ch)[0]
    img = split_projections(p, out)[0 if row_tx else 1]

    # analytic two-way delay written out by hand:
    lat, z, ref = grid_axes(cfg.grid_xz if row_tx else cfg.grid_yz)
    theta = (cfg.row_tx_angles if row_tx else cfg.col_tx_angles)[k]
    lat_j = elem_pos(j, cfg.n_cols if row_tx else cfg.n_rows, cfg.pitch)
    LAT, Z = np.meshgrid(lat, z, indexing="ij")
    tau = cfg.t0[e] + (Z * math.cos(theta) + ref * math.sin(theta)) / cfg.c \
        + np.sqrt((LAT - lat_j) ** 2 + Z ** 2) / cfg.c
    u = (tau - cfg.t_start) * cfg.fs
    tri = np.maximum(0.0, 1.0 - np.abs(u - n_s))                      # linear-interpolation kernel
    n = np.floor(u)
    tri = np.where((n >= 0) & (n + 1 <= cfg.n_samples - 1), tri, 0.0)  # edge rule (A6)
    expect = amp * tri * np.exp(1j * TWO_PI * cfg.fc * tau)
    if n_s not in (0, n_samples - 1):
        assert np.count_nonzero(tri) >= 3, "test geometry must hit the impulse"
    # the edge rule must actually exclude pixels in the edge cases
    assert (n_s not in (0, 1)) or np.any(n < 0)
    assert (n_s < n_samples - 2) or np.any(n + 1 > n_samples - 1)
    np.testing.assert_allclose(img, expect, rtol=0, atol=1e-9 * abs(amp))
    # every other output (other image) is exactly zero
    other = split_projections(p, out)[1 if row_tx else 0]
    assert np.all(other == 0)


def test_p1_impulse_is_seen():
    """The P1 geometry really does put pixels under the impulse (guards against a vacuous P1)."""
    cfg = tiny()
    p = params(cfg)
    ch = np.zeros(cfg.channel_shape, dtype=np.int16)
    ch[0, 2, rx_channel(cfg, True, 5), 160] = (1000, 0)
    img = split_projections(p, oracle.beamform(p, ch)[0])[0]
    assert np.count_nonzero(img) >= 5


# ---------------------------------------------------------------------------------------------
# P2  phase convention and absence of normalisation
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("f_number", [0.0, 1.2])
def test_p2_matched_phase_sums_coherently(f_number):
    cfg = tiny(f_number=f_number)
    rng = np.random.default_rng(5)
    win = rng.uniform(0.2, 1.0, cfg.n_cols + cfg.n_rows)
    p = params(cfg, elem_window=list(win))
    A = 20000.0
    for row_tx in (True, False):
        lat, z, ref = grid_axes(cfg.grid_xz if row_tx else cfg.grid_yz)
        il, iz = (7, 23) if row_tx else (3, 19)
        angles = cfg.row_tx_angles if row_tx else cfg.col_tx_angles
        n_el = cfg.n_cols if row_tx else cfg.n_rows
        ch = np.zeros(cfg.channel_shape, dtype=np.int16)
        wsum = 0.0
        for k, th in enumerate(angles):
            e = k if row_tx else len(cfg.row_tx_angles) + k
            for j in range(n_el):
                lat_j = elem_pos(j, n_el, cfg.pitch)
                tau = cfg.t0[e] + (z[iz] * math.cos(th) + ref * math.sin(th)) / cfg.c \
                    + math.hypot(lat[il] - lat_j, z[iz]) / cfg.c
                v = A * np.exp(-1j * TWO_PI * cfg.fc * tau)       # constant-envelope echo of the pixel
                ch[0, e, rx_channel(cfg, row_tx, j), :, 0] = int(round(v.real))
                ch[0, e, rx_channel(cfg, row_tx, j), :, 1] = int(round(v.imag))
                inside = f_number == 0.0 or abs(lat[il] - lat_j) <= z[iz] / (2 * f_number)
                wsum += (win[j] if row_tx else win[cfg.n_cols + j]) * inside
        img = split_projections(p, oracle.beamform(p, ch)[0])[0 if row_tx else 1]
        got = img[il, iz]
        expect = A * wsum                     # K * sum_j w_j, real and positive, NOT divided by anything
        assert abs(got - expect) <= 2e-4 * expect, (got, expect)   # int16 rounding of the echo only
        assert abs(got) >= np.abs(img).max() * (1 - 1e-9)          # and it is the image maximum


def test_p2_f_number_mask_counts_over_a_whole_grid():
    """w_j = [|lat - lat_j| <= z / (2 F#)], decided in fp64, edge inclusive.  With fc = 0 the
    rotation is 1 and constant IQ data A makes every term contribute exactly A, so P(lat, z) = A * K * (number of
    in-mask elements): the oracle's count is compared, over every pixel of both grids, with the inequality written
    out here.  F# is chosen so that one (pixel, element) pair sits 1e-10 (relative) INSIDE the edge, then 1e-10
    OUTSIDE: a decision taken in fp32, on rounded coordinates or with the wrong side / strictness miscounts it."""
    cfg = tiny(t0=None, t_start=0.0)
    A = 1000
    ch = np.zeros(cfg.channel_shape, dtype=np.int16)
    ch[..., 0] = A
    rng = np.random.default_rng(12)
    for trial in range(12):
        row_tx = trial % 2 == 0
        g = cfg.grid_xz if row_tx else cfg.grid_yz
        lat, z, _ = grid_axes(g)
        n_el = cfg.n_cols if row_tx else cfg.n_rows
        lat_j = elem_pos(np.arange(n_el), n_el, cfg.pitch)
        il, iz, j = int(rng.integers(g[0])), int(rng.integers(g[3])), int(rng.integers(n_el))
        dx = abs(lat[il] - lat_j[j])
        if dx < 1e-5:
            continue
        for side in (-1.0, +1.0):
            f_number = z[iz] / (2.0 * dx) * (1.0 + side * 1e-10)     # side < 0: the pair is just inside
            p = params(cfg, fc=0.0, f_number=f_number)
            out = oracle.beamform(p, ch)[0]
            for rt, img in zip((True, False), split_projections(p, out)):
                gg = cfg.grid_xz if rt else cfg.grid_yz
                la, zz, _ = grid_axes(gg)
                ne = cfg.n_cols if rt else cfg.n_rows
                lj = elem_pos(np.arange(ne), ne, cfg.pitch)
                K = len(cfg.row_tx_angles if rt else cfg.col_tx_angles)
                inside = np.abs(la[:, None, None] - lj[None, None, :]) <= zz[None, :, None] / (2.0 * f_number)
                count = inside.sum(-1)
                np.testing.assert_allclose(img, A * K * count, rtol=0, atol=1e-9)
                if rt == row_tx:
                    assert bool(inside[il, iz, j]) == (side < 0)
    # the edge itself is inclusive: power-of-two coordinates make |lat - lat_j| = z / (2 F#) exact
    g2 = (9, -4 * 2.0 ** -12, 2.0 ** -12, 8, 2.0 ** -7, 2.0 ** -12, 0.0)
    cfg2 = tiny(t0=None, t_start=0.0, pitch=2.0 ** -12, grid_xz=g2, grid_yz=g2, n_rows=9, n_cols=9)
    ch2 = np.zeros(cfg2.channel_shape, dtype=np.int16)
    ch2[..., 0] = A
    p2 = params(cfg2, fc=0.0, f_number=4.0)
    img = split_projections(p2, oracle.beamform(p2, ch2)[0])[0]
    la, zz, _ = grid_axes(g2)
    lj = elem_pos(np.arange(9), 9, cfg2.pitch)
    inside = np.abs(la[:, None, None] - lj[None, None, :]) <= zz[None, :, None] / 8.0
    on_edge = np.abs(la[:, None, None] - lj[None, None, :]) == zz[None, :, None] / 8.0
    assert on_edge.sum() >= 4                                        # the case really has pairs on the edge
    np.testing.assert_allclose(img, A * len(cfg2.row_tx_angles) * inside.sum(-1), rtol=0, atol=1e-9)


# ---------------------------------------------------------------------------------------------
# P3  demodulation of a pure tone at fc
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("fs,fc", [(20e6, 5e6), (40e6, 5e6), (25e6, 5e6), (20e6, 5.21e6)])
def test_p3_tone_demodulates_to_its_phasor(fs, fc):
    cfg = tiny(input_kind=0, fs=fs, n_samples=600, t_start=0.37e-6)
    p = params(cfg, fc=fc)
    A, phi = 9000.0, 0.7
    t = cfg.t_start + np.arange(cfg.n_samples) / fs
    rf = np.round(A * np.cos(TWO_PI * fc * t + phi)).astype(np.int16)
    iq = oracle.demod_channel(p, rf)
    L = (len(oracle.fir_taps(p)) - 1) // 2
    interior = iq[L:-L]
    # pass-band gain 1 at DC of the baseband, image at -2fc suppressed by the low-pass:
    # measured ripple of the specified 4*round(fs/fc)+1-tap Hamming design is < 0.5 %
    np.testing.assert_allclose(interior, A * np.exp(1j * phi), rtol=0, atol=5e-3 * A)
    assert abs(np.mean(interior) - A * np.exp(1j * phi)) < 2e-3 * A


def test_p3_fir_is_symmetric_lowpass_with_unit_dc_gain():
    cfg = tiny(input_kind=0)
    p = params(cfg)
    h = oracle.fir_taps(p)
    assert len(h) == 4 * round(cfg.fs / cfg.fc) + 1 == 17
    assert abs(h.sum() - 1.0) < 1e-14
    np.testing.assert_allclose(h, h[::-1], atol=1e-16)
    H = np.abs(np.fft.rfft(h, 4096))
    f = np.fft.rfftfreq(4096, 1.0 / cfg.fs)
    assert H[f <= 0.2 * cfg.fc].min() > 0.98          # pass band (baseband of a 65 % bandwidth pulse)
    assert H[f >= 2.0 * cfg.fc - 0.35 * cfg.fc].max() < 0.02   # mixer image around 2 fc
    p33 = params(tiny(input_kind=0, fs=40e6))
    assert len(oracle.fir_taps(p33)) == 33
    assert len(oracle.fir_taps(params(cfg, demod_taps=9))) == 9


# the 17 taps at fs = 4 fc, m = 0..8 (h[-m] = h[m]), written out: Hamming-windowed sinc(m/2), normalised to sum 1
# (SURVEY 8(c) step 0).  A Hann (0.5/0.5) or Blackman window, a sinc of the wrong argument or a missing
# normalisation changes the 3rd digit of several of them.
H17_HALF = [0.5008702925771573, 0.3076987787367444, 0.0, -0.07610584574867356, 0.0, 0.023211101786365082, 0.0,
            -0.005239181063014528, 0.0]


def test_p3_fir_taps_literal_and_library_cross_check():
    """ulm_oracle_fir against numbers stated here and against numpy's own sinc / hamming (a library routine, not the
    oracle's code): 17 taps (fs = 4 fc), 33 taps (fs = 8 fc), 21 taps (fs = 5 fc), and explicit tap counts."""
    cfg = tiny(input_kind=0)
    h = oracle.fir_taps(params(cfg))
    np.testing.assert_allclose(h[8:], H17_HALF, rtol=0, atol=1e-15)
    np.testing.assert_allclose(h[:9][::-1], H17_HALF, rtol=0, atol=1e-15)
    for fs, fc, taps, L in [(20e6, 5e6, 0, 8), (40e6, 5e6, 0, 16), (25e6, 5e6, 0, 10), (20e6, 5e6, 9, 4),
                            (40e6, 5.21e6, 25, 12), (20e6, 5.21e6, 0, 8)]:
        hh = oracle.fir_taps(params(tiny(input_kind=0, fs=fs), fc=fc, demod_taps=taps))
        m = np.arange(-L, L + 1)
        ref = np.sinc(2.0 * fc * m / fs) * np.hamming(2 * L + 1)
        ref /= ref.sum()
        assert len(hh) == 2 * L + 1
        np.testing.assert_allclose(hh, ref, rtol=0, atol=1e-15)


def test_p3_impulse_response_and_zero_padding():
    """rf = delta at n0  ->  iq[n] = 2 h[n-n0] exp(-j 2 pi fc t_n0); near the record ends the
    missing samples count as zero (no wrap-around, no renormalisation)."""
    cfg = tiny(input_kind=0, n_samples=64, t_start=0.2e-6)
    p = params(cfg)
    h = oracle.fir_taps(p)
    L = (len(h) - 1) // 2
    for n0 in (0, 3, 31, 63):
        rf = np.zeros(cfg.n_samples, dtype=np.int16)
        rf[n0] = 1000
        iq = oracle.demod_channel(p, rf)
        expect = np.zeros(cfg.n_samples, dtype=complex)
        for n in range(cfg.n_samples):
            m = n - n0
            if -L <= m <= L:
                expect[n] = 2 * h[m + L] * 1000 * np.exp(-1j * TWO_PI * cfg.fc * (cfg.t_start + n0 / cfg.fs))
        np.testing.assert_allclose(iq, expect, atol=1e-9)


# ---------------------------------------------------------------------------------------------
# P4  brute-force 3-D DAS (independently coded, point-outer) == projection on the reference plane
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("input_kind", [0, 1])
def test_p4_volume_reference_planes_equal_projections(input_kind):
    cfg = tiny(input_kind=input_kind, f_number=1.3)
    rng = np.random.default_rng(11)
    win = list(rng.uniform(0.1, 1.0, cfg.n_cols + cfg.n_rows))
    p = params(cfg, elem_window=win)
    ch = synth.random_channel(cfg, 1, seed=3, amplitude=3000)
    out = oracle.beamform(p, ch)[0]
    p_xz, p_yz = split_projections(p, out)
    x, z_xz, y_ref = grid_axes(cfg.grid_xz)
    y, z_yz, x_ref = grid_axes(cfg.grid_yz)
    # XZ projection == plane y = y_ref of the row-tx (RC) volume
    v_rc, v_cr = oracle.volume(p, ch[0], x, [y_ref - 1e-3, y_ref, y_ref + 0.5e-3], z_xz)
    scale = np.abs(p_xz).max()
    np.testing.assert_allclose(v_rc[:, 1, :], p_xz, rtol=0, atol=1e-11 * scale)
    assert np.abs(v_rc[:, 0, :] - p_xz).max() > 1e-3 * scale      # other planes differ (steered tx)
    # YZ projection == plane x = x_ref of the column-tx (CR) volume
    v_rc2, v_cr2 = oracle.volume(p, ch[0], [x_ref, x_ref + 0.7e-3], y, z_yz)
    np.testing.assert_allclose(v_cr2[0], p_yz, rtol=0, atol=1e-11 * np.abs(p_yz).max())
    assert np.abs(v_cr2[1] - p_yz).max() > 1e-3 * np.abs(p_yz).max()


def test_p4_compound0_slices_sum_to_compound1():
    cfg = tiny(input_kind=0)
    ch = synth.random_channel(cfg, 2, seed=9)
    p1, p0 = params(cfg), params(cfg, compound=0)
    o1, o0 = oracle.beamform(p1, ch), oracle.beamform(p0, ch)
    nxz = cfg.grid_xz[0] * cfg.grid_xz[3]
    nyz = cfg.grid_yz[0] * cfg.grid_yz[3]
    kr, kc = len(cfg.row_tx_angles), len(cfg.col_tx_angles)
    assert o0.shape[1] == kr * nxz + kc * nyz
    for f in range(2):
        sxz = o0[f, :kr * nxz].reshape(kr, nxz).sum(0)
        syz = o0[f, kr * nxz:].reshape(kc, nyz).sum(0)
        np.testing.assert_allclose(sxz, o1[f, :nxz], atol=1e-9 * np.abs(o1).max())
        np.testing.assert_allclose(syz, o1[f, nxz:], atol=1e-9 * np.abs(o1).max())


# ---------------------------------------------------------------------------------------------
# P5  linearity
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("input_kind", [0, 1])
def test_p5_linearity(input_kind):
    cfg = tiny(input_kind=input_kind, f_number=1.5)
    p = params(cfg)
    a = synth.random_channel(cfg, 1, seed=1, amplitude=8000)
    b = synth.random_channel(cfg, 1, seed=2, amplitude=8000)
    Ba, Bb, Bab, Bna = (oracle.beamform(p, v) for v in (a, b, a + b, -a))
    s = np.abs(Bab).max()
    assert s > 0
    assert np.abs(Bab - (Ba + Bb)).max() <= 1e-12 * s
    assert np.abs(Bna + Ba).max() <= 1e-12 * s
    assert np.all(oracle.beamform(p, np.zeros_like(a)) == 0)


# ---------------------------------------------------------------------------------------------
# P7  a point scatterer on the reference plane peaks within one pixel of its position (RF input,
#     noise, other scatterers present) -- geometry end to end through the echo simulator
# ---------------------------------------------------------------------------------------------
def test_p7_point_scatterer_peak():
    cfg = synth.config(0).with_(n_frames=1)
    main = np.array([[1.31e-3, 0.0, 11.7e-3, 1.0]])        # on y_ref = 0
    rng = np.random.default_rng(2)
    others = np.column_stack([rng.uniform(-4e-3, 4e-3, 6), rng.uniform(2e-3, 4e-3, 6),
                              rng.uniform(6e-3, 19e-3, 6), np.full(6, 0.05)])
    ch = synth.render(cfg, [0], noise=True, scat={0: np.concatenate([main, others])})
    p = params(cfg)
    p_xz, p_yz = split_projections(p, oracle.beamform(p, ch)[0])
    x, z, _ = grid_axes(cfg.grid_xz)
    il, iz = np.unravel_index(np.argmax(np.abs(p_xz)), p_xz.shape)
    assert abs(x[il] - main[0, 0]) <= cfg.grid_xz[2] and abs(z[iz] - main[0, 2]) <= cfg.grid_xz[5]
    # the same scatterer seen in the YZ image of a scene mirrored onto x_ref = 0
    main_t = main[:, [1, 0, 2, 3]]
    main_t[0, 1] = -2.05e-3
    ch = synth.render(cfg, [0], noise=True, scat={0: main_t})
    p_xz, p_yz = split_projections(p, oracle.beamform(p, ch)[0])
    y, z, _ = grid_axes(cfg.grid_yz)
    il, iz = np.unravel_index(np.argmax(np.abs(p_yz)), p_yz.shape)
    assert abs(y[il] - main_t[0, 1]) <= cfg.grid_yz[2] and abs(z[iz] - main_t[0, 2]) <= cfg.grid_yz[5]


def test_p7_steered_single_angle_off_plane():
    """compound=0: with one steered angle the slice through y_ref still focuses a scatterer that sits
    OFF the plane, displaced axially by about (y0 - y_ref) tan(theta/2)-like amounts (PAPER.md:45,
    "rigid axial shift determined by the transmit steering angle"); the lateral position is kept."""
    d = synth.LAMBDA_M / 2
    g = centred_grid(24, d, 160, 11.0e-3, d / 8)
    cfg = synth.config(0).with_(n_frames=1, grid_xz=g)
    y0 = 3.0e-3
    sc = np.array([[0.9e-3, y0, 12.0e-3, 1.0]])
    ch = synth.render(cfg, [0], noise=False, scat={0: sc})
    p = params(cfg, compound=0)
    out = oracle.beamform(p, ch)[0]
    nxz = cfg.grid_xz[0] * cfg.grid_xz[3]
    x, z, _ = grid_axes(cfg.grid_xz)
    peaks = []
    for k, th in enumerate(cfg.row_tx_angles):
        img = out[k * nxz:(k + 1) * nxz].reshape(cfg.grid_xz[0], cfg.grid_xz[3])
        il, iz = np.unravel_index(np.argmax(np.abs(img)), img.shape)
        assert abs(x[il] - sc[0, 0]) <= cfg.grid_xz[2]
        peaks.append(z[iz])
        # first-order prediction of the apparent depth: the tx path gains y0 sin(theta), shared
        # between the two legs of a near-axial echo
        z_pred = sc[0, 2] + y0 * math.sin(th) / (math.cos(th) + 1.0)
        assert abs(z[iz] - z_pred) <= 0.04e-3, (k, z[iz], z_pred)
    assert peaks[0] < peaks[1] < peaks[2]


# ---------------------------------------------------------------------------------------------
# P8  symmetries
# ---------------------------------------------------------------------------------------------
def _sym_cfg(**kw):
    d = synth.LAMBDA_M / 2
    ang = tuple(np.radians([-5.0, 2.0, 6.0]))
    g = centred_grid(14, d, 16, 6e-3, d, ref=0.35e-3)
    return tiny(row_tx_angles=ang, col_tx_angles=ang, grid_xz=g, grid_yz=g,
                t0=(1e-7, -2e-7, 3e-7, 1e-7, -2e-7, 3e-7), **kw)


@pytest.mark.parametrize("input_kind", [0, 1])
def test_p8_transpose_swaps_projections(input_kind):
    cfg = _sym_cfg(input_kind=input_kind)
    p = params(cfg)
    ch = synth.random_channel(cfg, 1, seed=21)
    kr, nr = len(cfg.row_tx_angles), cfg.n_rows
    # swap the roles of rows and columns: row-tx events <-> column-tx events, row channels <-> columns
    sw = np.concatenate([ch[:, kr:], ch[:, :kr]], axis=1)
    sw = np.concatenate([sw[:, :, nr:], sw[:, :, :nr]], axis=2)
    a_xz, a_yz = split_projections(p, oracle.beamform(p, ch)[0])
    b_xz, b_yz = split_projections(p, oracle.beamform(p, sw)[0])
    s = np.abs(a_xz).max()
    np.testing.assert_allclose(b_xz, a_yz, atol=1e-12 * s)
    np.testing.assert_allclose(b_yz, a_xz, atol=1e-12 * s)
    assert np.abs(a_xz - a_yz).max() > 1e-3 * s


def test_p8_mirror_x():
    cfg = _sym_cfg()
    p = params(cfg)
    ch = synth.random_channel(cfg, 1, seed=22)
    nr = cfg.n_rows
    mir = ch.copy()
    mir[:, :, nr:] = ch[:, :, nr:][:, :, ::-1]            # reverse the column (x-indexed) channels
    a_xz, a_yz = split_projections(p, oracle.beamform(p, ch)[0])
    # the lateral grid is symmetric about 0, so mirroring x is a flip of the lateral index
    m_xz, _ = split_projections(p, oracle.beamform(p, mir)[0])
    np.testing.assert_allclose(m_xz, a_xz[::-1], atol=1e-12 * np.abs(a_xz).max())
    # same statement with an explicitly reversed (negative-step) lateral grid and the original order
    g = cfg.grid_xz
    g_rev = (g[0], g[1] + (g[0] - 1) * g[2], -g[2]) + g[3:]
    p_rev = params(cfg, grid_xz=g_rev)
    r_xz, _ = split_projections(p_rev, oracle.beamform(p_rev, ch)[0])
    np.testing.assert_allclose(r_xz, a_xz[::-1], atol=1e-12 * np.abs(a_xz).max())


def test_p8_time_shift_invariance():
    cfg = _sym_cfg(input_kind=1)
    d = 9
    ch = np.zeros(cfg.channel_shape, dtype=np.int16)
    rng = np.random.default_rng(4)
    ch[..., 40:420, :] = rng.integers(-5000, 5000, size=ch[..., 40:420, :].shape)
    sh = np.zeros_like(ch)
    sh[..., 40 + d:420 + d, :] = ch[..., 40:420, :]       # every record delayed by d samples ...
    p_a = params(cfg)
    p_b = params(cfg, t_start=cfg.t_start - d / cfg.fs)   # ... and the clock started d samples earlier
    a, b = oracle.beamform(p_a, ch), oracle.beamform(p_b, sh)
    assert np.abs(a).max() > 0
    np.testing.assert_allclose(b, a, atol=1e-9 * np.abs(a).max())


def test_p8_orthogonal_only_layout_matches_full_layout():
    """A8: only the aperture orthogonal to the transmitting one is read."""
    cfg = _sym_cfg(input_kind=0)
    ch = synth.random_channel(cfg, 1, seed=30)
    kr, nr = len(cfg.row_tx_angles), cfg.n_rows
    ortho = np.concatenate([ch[:, :kr, nr:], ch[:, kr:, :nr]], axis=1)
    poison = ch.copy()
    poison[:, :kr, :nr] = 31000                            # same-aperture channels must be ignored
    poison[:, kr:, nr:] = -31000
    p_full = params(cfg)
    p_orth = params(cfg.with_(all_channels=False))
    a = oracle.beamform(p_full, ch)
    np.testing.assert_array_equal(oracle.beamform(p_full, poison), a)
    np.testing.assert_array_equal(oracle.beamform(p_orth, ortho), a)


# ---------------------------------------------------------------------------------------------
# P9  work count
# ---------------------------------------------------------------------------------------------
def test_p9_work_counts():
    c0, c1, c2, c3, c4 = (synth.config(i) for i in range(5))
    assert c0.gather_samples_per_frame() * c0.n_frames == 2_359_296
    assert c1.gather_samples_per_frame() == 83_128_320
    assert c2.gather_samples_per_frame() * c2.n_frames == 24_938_496_000
    assert c3.gather_samples_per_frame() * c3.n_frames == 99_753_984_000
    assert c4.gather_samples_per_frame() == 180 * c1.gather_samples_per_frame()
    assert np.prod(c2.channel_shape) * 2 == 6_920_601_600          # "~6.9 GB int16"
    assert (c1.grid_xz[0], c1.grid_xz[3]) == (180, 164) and (c3.grid_xz[0], c3.grid_xz[3]) == (360, 328)
    assert (c0.grid_xz[0], c0.grid_xz[3]) == (64, 96)
    for c in (c1, c3):                                             # 25 x 27.4 x 27.4 mm^3 volume
        assert abs(c.grid_xz[3] * c.grid_xz[5] - 25e-3) < 0.5e-3
        assert abs(c.grid_xz[0] * c.grid_xz[2] - 27.4e-3) < 0.5e-3
        assert abs(c.n_cols * c.pitch - 27.4e-3) < 0.1e-3


def test_touched_sample_range_is_inside_the_record():
    """A11: every pixel/element/angle of configs 0, 1, 3 reads samples inside [0, Ns-1]."""
    for idx in (0, 1, 3):
        cfg = synth.config(idx)
        x, z, ref = grid_axes(cfg.grid_xz)
        xj = elem_pos(np.arange(cfg.n_cols), cfg.n_cols, cfg.pitch)
        th = np.array(cfg.row_tx_angles)
        dmax = np.abs(x[:, None] - xj[None, :]).max()
        u_min = (z[0] * np.cos(th).min() + z[0]) / cfg.c * cfg.fs
        u_max = (z[-1] + math.hypot(dmax, z[-1])) / cfg.c * cfg.fs
        assert u_min > 16 and u_max < cfg.n_samples - 17


def test_golden_fixture_unchanged():
    """The oracle still reproduces tests/golden/tiny_projection.txt (written by make_golden.py)."""
    import importlib.util
    import os
    here = os.path.dirname(os.path.abspath(__file__))
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(here, "golden", "make_golden.py"))
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
    cfg, ch, win = mg.golden_case()
    out = oracle.beamform(params(cfg, elem_window=win), ch)[0]
    ref = np.loadtxt(os.path.join(here, "golden", "tiny_projection.txt"))
    np.testing.assert_allclose(out, ref[:, 0] + 1j * ref[:, 1], rtol=1e-13, atol=1e-9)

"""GPU parity: the CUDA path (through the C-ABI) against the fp64 oracle, element by element, on the
same seeded inputs.  Bar (BASELINE.json north_star): max|gpu - oracle| <= 1e-4 * max|oracle| per frame,
taken over both projections of the frame jointly."""
import math

import numpy as np
import pytest

import oracle
import synth
from helpers import assert_mask_margin, mask_margin, rel_err, rounded_kwargs
from synth import centred_grid

pytestmark = pytest.mark.gpu

TOL = 1e-4
# White-noise channel data is the stress case of the scratch formats: it has no coherent echo, so the image maximum is
# an incoherent sum and a per-term format error is measured against a maximum ~sqrt(N) times smaller than on echo
# data, and (through the library's own low-pass) |d| / |iq| is 0.85 instead of ~0.3.  Every white-noise case is checked
# against the same oracle result with full entries (precision = 2) at NOISE_TOL_FULL -- sharp enough to expose any
# planning / indexing / edge error -- and with the entries the plan selects by DEFAULT (precision = 0: compact entries
# with the two-term interpolation weight for RF input, full entries for IQ input) at the north-star bar TOL.
# Only the opt-in fast format (precision = 1: fp16 interpolation weight, documented in ulm_rca.h as holding 1e-4 on
# band-limited echo data only) is allowed its format bound NOISE_TOL_FAST on white noise.
NOISE_TOL_FULL = 2e-5
NOISE_TOL_FAST = 1.5e-4


def tol_of(info):
    return {1: NOISE_TOL_FAST, 2: NOISE_TOL_FULL, 3: TOL}[info["precision"]]


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2511_21647_b200 import build
    build.build()
    return torch


def run_pair(torch, cfg, ch, plan_extra=None, **overrides):
    """Beamform `ch` with the oracle and with the CUDA plan built from the same rounded arguments."""
    from paper_2511_21647_b200 import Plan
    kw = rounded_kwargs(cfg, **overrides)
    assert_mask_margin(kw)      # f-number cases: no pair within fp32 rounding of the mask edge (oracle decides in fp64)
    ref = oracle.beamform(oracle.OracleParams(**kw), ch)
    with Plan(**kw, **(plan_extra or {})) as plan:
        d_ch = torch.from_numpy(np.ascontiguousarray(ch)).cuda()
        out = plan.beamform(d_ch)
        torch.cuda.synchronize()
        info = plan.info()
    return out.cpu().numpy(), ref, info


def run_gpu(torch, kw, ch, plan_extra=None):
    from paper_2511_21647_b200 import Plan
    with Plan(**kw, **(plan_extra or {})) as plan:
        out = plan.beamform(torch.from_numpy(np.ascontiguousarray(ch)).cuda())
        torch.cuda.synchronize()
        info = plan.info()
    return out.cpu().numpy(), info


def check_noise(torch, cfg, ch, plan_extra=None, **overrides):
    """White-noise input: full entries at NOISE_TOL_FULL, then the requested plan at its format bound."""
    kw = rounded_kwargs(cfg, **overrides)
    assert_mask_margin(kw)
    ref = oracle.beamform(oracle.OracleParams(**kw), ch)
    extra = dict(plan_extra or {})
    full, info_full = run_gpu(torch, kw, ch, dict(extra, precision=2))
    assert info_full["precision"] == 2
    assert_parity(full, ref, tol=NOISE_TOL_FULL)
    gpu, info = run_gpu(torch, kw, ch, extra)
    assert_parity(gpu, ref, tol=tol_of(info))
    return gpu, ref, info


def assert_parity(gpu, ref, tol=TOL):
    assert gpu.shape == ref.shape
    errs = [rel_err(gpu[f], ref[f]) for f in range(ref.shape[0])]
    worst = max(errs) if errs else 0.0
    print("PARITY worst max|gpu-oracle|/max|oracle| = %.3e over %d frame(s)" % (worst, len(errs)))
    for f, e in enumerate(errs):
        assert e <= tol, "frame %d: max|gpu-oracle|/max|oracle| = %.3e > %.1e" % (f, e, tol)
    return worst


def small(**kw):
    """24+20-element array (n_rows != n_cols), 3+2 angles, grids that span several tiles and a ragged tail."""
    d = synth.LAMBDA_M / 2
    base = dict(n_rows=24, n_cols=20, pitch=0.3e-3, n_samples=700,
                row_tx_angles=tuple(np.radians([-7.0, 1.0, 6.0])), col_tx_angles=tuple(np.radians([-4.0, 8.0])),
                grid_xz=centred_grid(37, d, 53, 6e-3, d, ref=0.4e-3),
                grid_yz=centred_grid(29, 1.2 * d, 41, 6.5e-3, 0.8 * d, ref=-0.3e-3),
                n_frames=3, t_start=0.9e-6, t0=(0.2e-6, -0.1e-6, 0.05e-6, 0.3e-6, -0.25e-6))
    base.update(kw)
    return synth.config(0).with_(**base)


KERNELS = [1, 0]     # generic gather kernel; auto (shared-memory ring kernel where it applies)


@pytest.mark.parametrize("kernel", KERNELS)
def test_config0_full(torch_cuda, kernel):
    cfg = synth.config(0)
    ch = synth.render(cfg)
    gpu, ref, info = run_pair(torch_cuda, cfg, ch, plan_extra=dict(kernel=kernel))
    worst = assert_parity(gpu, ref)
    assert info["events_executed"] == 4       # the +-5 degree events of each aperture fold (centred slices, t0 = 0)
    print("cfg0 kernel=%d worst rel err %.3e  info %s" % (info["kernel"], worst, info))


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("case", ["rf", "rf_full", "iq", "iq_bandlimited_compact", "apod", "orth", "fs25", "neg_dlat",
                                  "taps9", "one_aperture", "t_start_odd", "fs40", "fs40_taps25", "fs40_edges"])
def test_small_variants(torch_cuda, kernel, case):
    extra = {}
    cfg = small()
    if case == "iq":
        cfg = small(input_kind=1)            # precision auto -> full entries (spectrum unknown)
    elif case == "rf_full":
        extra = dict(precision=2)
    elif case == "iq_bandlimited_compact":
        cfg = small(input_kind=1)
        extra = dict(precision=1)
    elif case == "apod":
        w = np.hanning(cfg.n_cols + 2)[1:-1].tolist() + np.hanning(cfg.n_rows + 2)[1:-1].tolist()
        cfg = small(f_number=1.5, elem_window=tuple(w))
    elif case == "orth":
        cfg = small(n_rows=20, n_cols=20, all_channels=False)
    elif case == "fs25":
        cfg = small(fs=25e6, fc=5.21e6)
    elif case == "neg_dlat":
        g = small().grid_xz
        cfg = small(grid_xz=(g[0], g[1] + (g[0] - 1) * g[2], -g[2]) + g[3:])
    elif case == "taps9":
        cfg = small(demod_taps=9)
    elif case == "one_aperture":
        cfg = small(col_tx_angles=(), t0=(0.2e-6, -0.1e-6, 0.05e-6))
    elif case == "t_start_odd":
        # fs = 4 fc with fc * t_start NOT a multiple of a quarter cycle: the quadrature pre-pass (analytic signal from
        # two real filters, no mixer) must still apply -- its entries carry the sample's own phase exactly
        cfg = small(t_start=0.937e-6)
    elif case == "fs40":
        # fs = 8 fc with the default 33 taps: the analytic pre-pass (two real filters, no mixer), t_start off the grid
        cfg = small(fs=40e6, n_samples=1400, t_start=0.913e-6)
    elif case == "fs40_taps25":
        cfg = small(fs=40e6, n_samples=1400, demod_taps=25)      # same sampling, other tap count: the generic path
    elif case == "fs40_edges":
        # records so short that the image runs past both ends: the zero padding of the filter and the edge rule
        g = small().grid_xz
        cfg = small(fs=40e6, n_samples=520, t_start=3.2e-6, grid_xz=g[:3] + (70, 2e-3, g[5], g[6]))
    ch = synth.random_channel(cfg, cfg.n_frames, seed=17, amplitude=6000)
    if case == "iq_bandlimited_compact":
        # the compact format is meant for band-limited IQ: smooth the white data along the sample axis
        k = np.array([1, 4, 6, 4, 1], dtype=np.float64) / 16
        sm = np.apply_along_axis(lambda v: np.convolve(v, k, mode="same"), -2, ch.astype(np.float64))
        ch = np.round(sm).astype(np.int16)
    gpu, ref, info = check_noise(torch_cuda, cfg, ch, plan_extra=dict(kernel=kernel, **extra))
    assert info["precision"] == (2 if case in ("iq", "rf_full") else 1 if case == "iq_bandlimited_compact" else 3)


@pytest.mark.parametrize("kernel", KERNELS)
def test_per_angle_slices(torch_cuda, kernel):
    """compound = 0: one slice per transmit event (the paper's S_k), through the generic kernel and
    through the ring kernel (one work item per angle and tile)."""
    cfg = small(compound=0)
    ch = synth.random_channel(cfg, 2, seed=5, amplitude=6000)
    _, _, info = check_noise(torch_cuda, cfg, ch, plan_extra=dict(kernel=kernel))
    assert info["kernel"] == (1 if kernel == 1 else 2)
    # 13 frames (a full 12-frame group + 1), f-number mask and window, a single-aperture plan
    w = np.hanning(cfg.n_cols + 2)[1:-1].tolist() + np.hanning(cfg.n_rows + 2)[1:-1].tolist()
    cfg13 = small(compound=0, n_frames=13, f_number=1.5, elem_window=tuple(w))
    check_noise(torch_cuda, cfg13, synth.random_channel(cfg13, 13, seed=6, amplitude=6000), plan_extra=dict(kernel=kernel))
    cfg1 = small(compound=0, col_tx_angles=(), t0=(0.2e-6, -0.1e-6, 0.05e-6))
    check_noise(torch_cuda, cfg1, synth.random_channel(cfg1, 3, seed=7, amplitude=6000), plan_extra=dict(kernel=kernel))
    # and the slices add up to the compounded images (full entries: the ring and the generic kernel differ by fp32
    # rounding only; with compact entries a delay that differs in the last fp32 bit can round the fp16 weight the
    # other way, so the two kernels agree to the format bound, not to 1e-5)
    nxz = cfg.grid_xz[0] * cfg.grid_xz[3]
    kr = len(cfg.row_tx_angles)
    for precision, bound in [(2, 1e-5), (3, TOL)]:
        kw = rounded_kwargs(cfg)
        gpu, _ = run_gpu(torch_cuda, kw, ch, dict(precision=precision, kernel=kernel))
        gpu1, info1 = run_gpu(torch_cuda, rounded_kwargs(cfg.with_(compound=1)), ch, dict(precision=precision))
        assert info1["kernel"] == 2
        s = gpu[:, :kr * nxz].reshape(2, kr, nxz).sum(1)
        assert np.abs(s - gpu1[:, :nxz]).max() <= bound * np.abs(gpu1).max()


@pytest.mark.parametrize("kernel", KERNELS)
def test_event_folding(torch_cuda, kernel):
    """Transmit events with identical reference-slice delays (mirror angles about a centred slice, equal t0) are
    added in the pre-pass and beamformed once; the oracle sums every event separately.  Folding must happen exactly
    when the delays coincide -- and the result must not depend on it."""
    d = synth.LAMBDA_M / 2
    gx, gy = centred_grid(37, d, 53, 6e-3, d, ref=0.0), centred_grid(29, 1.2 * d, 41, 6.5e-3, 0.8 * d, ref=0.0)
    mirror = tuple(np.radians([-6.0, 2.0, 6.0]))
    cases = [
        # (overrides, events executed): the +-6 degree pair of the row-tx aperture folds, nothing else does
        (dict(grid_xz=gx, grid_yz=gy, row_tx_angles=mirror, t0=(0.1e-6, -0.1e-6, 0.1e-6, 0.3e-6, -0.25e-6)), 4),
        # a centred slice but different t0 inside the pair: no folding
        (dict(grid_xz=gx, grid_yz=gy, row_tx_angles=mirror, t0=(0.1e-6, -0.1e-6, 0.2e-6, 0.3e-6, -0.25e-6)), 5),
        # equal t0 but an off-centre reference slice (ref sin(theta) differs in sign): no folding
        (dict(row_tx_angles=mirror, t0=(0.1e-6, -0.1e-6, 0.1e-6, 0.3e-6, -0.25e-6)), 5),
        # both apertures fold, one of them to a single event; duplicated angles fold too; f-number mask + window
        (dict(grid_xz=gx, grid_yz=gy, row_tx_angles=tuple(np.radians([-3.0, 3.0])),
              col_tx_angles=tuple(np.radians([5.0, 0.0, 0.0, -5.0])), t0=None, f_number=1.5,
              elem_window=tuple(np.hanning(22)[1:-1].tolist() + np.hanning(26)[1:-1].tolist())), 3),
        # the generic pre-pass (fs != 4 fc) and IQ input add the folded records too; 13 frames = a full 12-frame group + 1
        (dict(grid_xz=gx, grid_yz=gy, row_tx_angles=mirror, t0=None, fs=25e6, fc=5.21e6, n_frames=13), 4),
        (dict(grid_xz=gx, grid_yz=gy, row_tx_angles=mirror, t0=None, input_kind=1), 4),
    ]
    for over, n_exec in cases:
        cfg = small(**over)
        ch = synth.random_channel(cfg, cfg.n_frames, seed=77, amplitude=6000)
        gpu, ref, info = check_noise(torch_cuda, cfg, ch, plan_extra=dict(kernel=kernel))
        assert info["events_executed"] == n_exec, (over, info)
    # folded events through batches of max_frames (11 frames in batches of 4)
    cfg = small(grid_xz=gx, grid_yz=gy, row_tx_angles=mirror, t0=None, n_frames=11)
    ch = synth.random_channel(cfg, 11, seed=79, amplitude=6000)
    gpu, ref, info = check_noise(torch_cuda, cfg, ch, plan_extra=dict(kernel=kernel, max_frames=4))
    assert info["events_executed"] == 4
    # per-angle output never folds
    cfg = small(grid_xz=gx, grid_yz=gy, row_tx_angles=mirror, t0=None, compound=0)
    ch = synth.random_channel(cfg, cfg.n_frames, seed=78, amplitude=6000)
    gpu, ref, info = check_noise(torch_cuda, cfg, ch)
    assert info["events_executed"] == 5


@pytest.mark.parametrize("kernel", KERNELS)
def test_batching_and_ragged_frame_counts(torch_cuda, kernel):
    """n_frames > max_frames is processed in batches; odd frame counts leave a ragged last group."""
    cfg = small(n_frames=11)
    ch = synth.random_channel(cfg, 11, seed=23, amplitude=6000)
    check_noise(torch_cuda, cfg, ch, plan_extra=dict(max_frames=4, kernel=kernel))
    check_noise(torch_cuda, cfg, ch[:1], plan_extra=dict(max_frames=4, kernel=kernel))


def test_plan_reuse_and_determinism(torch_cuda):
    """One plan, calls of different sizes in turn (4-frame and 12-frame scratch groups alternate, batches of
    max_frames), every call repeated: results are bitwise reproducible (no atomics anywhere on the path) and do not
    depend on what the scratch held before."""
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    cfg = small(n_frames=17)
    ch = torch.from_numpy(synth.random_channel(cfg, 17, seed=91, amplitude=6000)).cuda()
    with Plan(**rounded_kwargs(cfg), max_frames=13) as plan:
        ref17 = plan.beamform(ch).cpu().numpy()
        for n in (3, 17, 1, 12, 13, 4, 17):
            a = plan.beamform(ch[:n]).cpu().numpy()
            b = plan.beamform(ch[:n]).cpu().numpy()
            np.testing.assert_array_equal(a, b)
            if n > 4:      # the same frames in the same 12-frame groups: identical arithmetic
                np.testing.assert_array_equal(a[:12], ref17[:12])
            else:
                # 4-frame groups.  With compact entries the low mantissa byte of a direct fp24 value is a byte of
                # another frame of its 4-frame chunk, so a frame's result depends, below
                # 2^-16 per term, on which frames share the chunk (here: frame 3 is absent): format level, not 0
                assert np.abs(a - ref17[:n]).max() <= 5e-5 * np.abs(ref17).max()


def test_two_live_plans_with_different_filters(torch_cuda):
    """Plans with different demodulation filters (default 17 taps, 25 taps, fs = 5 fc with 21 taps) are alive at the same
    time and used in turn, on two streams: each keeps its own constants (they travel in the kernel parameters)."""
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    cfgs = [small(n_frames=3), small(n_frames=3, demod_taps=25), small(n_frames=3, fs=25e6)]
    kws = [rounded_kwargs(c) for c in cfgs]
    chs = [synth.random_channel(c, 3, seed=70 + i, amplitude=6000) for i, c in enumerate(cfgs)]
    refs = [oracle.beamform(oracle.OracleParams(**kw), ch) for kw, ch in zip(kws, chs)]
    plans = [Plan(**kw, precision=2) for kw in kws]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    try:
        d_chs = [torch.from_numpy(ch).cuda() for ch in chs]
        torch.cuda.synchronize()
        outs = [None] * len(plans)
        for rep in range(2):
            for i in (2, 0, 1):
                outs[i] = plans[i].beamform(d_chs[i], stream=streams[i % 2])
        torch.cuda.synchronize()
        for out, ref in zip(outs, refs):
            assert_parity(out.cpu().numpy(), ref, tol=NOISE_TOL_FULL)
    finally:
        for plan in plans:
            plan.close()


def test_plans_on_two_host_threads_and_two_devices(torch_cuda):
    """ulm_rca.h: different plans may be in flight at the same time, on any devices.  Two host threads each create,
    use and destroy their own plan concurrently (kernel attributes are set per plan / device, not once per process);
    with two or more GPUs the second thread works on cuda:1, otherwise both share cuda:0.  A tensor on another
    device than the plan's is refused by the binding."""
    import threading
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    n_dev = torch.cuda.device_count()
    cfg = small(n_frames=13)
    kw = rounded_kwargs(cfg)
    chs = [synth.random_channel(cfg, 13, seed=200 + i, amplitude=6000) for i in range(2)]
    refs = [oracle.beamform(oracle.OracleParams(**kw), ch) for ch in chs]
    outs, errs = [None, None], []

    def work(i):
        try:
            dev = i % n_dev
            torch.cuda.set_device(dev)
            for _ in range(3):
                with Plan(**kw) as plan:
                    out = plan.beamform(torch.from_numpy(chs[i]).to("cuda:%d" % dev), stream=torch.cuda.Stream(dev))
                    torch.cuda.synchronize(dev)
                    outs[i] = out.cpu().numpy()
        except Exception as exc:        # surfaced in the main thread
            errs.append(exc)

    threads = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    for th in threads:
        th.start()
    for th in threads:
        th.join()
    torch.cuda.set_device(0)
    assert not errs, errs
    for out, ref in zip(outs, refs):
        assert_parity(out, ref, tol=TOL)
    if n_dev >= 2:
        with Plan(**kw) as plan:
            with pytest.raises(ValueError):
                plan.beamform(torch.from_numpy(chs[0]).to("cuda:1"))


def test_zero_frames_and_bad_buffers(torch_cuda):
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    cfg = small()
    with Plan(**rounded_kwargs(cfg)) as plan:
        empty = torch.empty((0,) + cfg.channel_shape[1:], dtype=torch.int16, device="cuda")
        out = plan.beamform(empty)
        assert out.shape[0] == 0
        with pytest.raises(ValueError):
            plan.beamform(torch.zeros((1, 3, 3), dtype=torch.int16, device="cuda"))
        with pytest.raises(Exception):
            plan.beamform_volume(torch.zeros((1,) + cfg.channel_shape[1:], dtype=torch.int16, device="cuda"))
        with pytest.raises(ValueError):
            plan.beamform_volume(torch.zeros((1, 3, 3), dtype=torch.int16, device="cuda"))
        with pytest.raises(ValueError):
            plan.beamform(torch.zeros((1,) + cfg.channel_shape[1:], dtype=torch.int16, device="cuda"),
                          out=torch.zeros(7, dtype=torch.complex64, device="cuda"))


def test_edge_rule_record_ends_inside_the_image(torch_cuda):
    """Records that start / end inside the imaged depth range: terms with n < 0 or n+1 > Ns-1 are dropped
    on both sides identically (data near the ends is non-zero)."""
    for t_start, ns in [(8.9e-6, 700), (0.9e-6, 230)]:
        cfg = small(t_start=t_start, n_samples=ns, input_kind=1)
        ch = synth.random_channel(cfg, 2, seed=31, amplitude=6000)
        gpu, ref, _ = run_pair(torch_cuda, cfg, ch)
        assert_parity(gpu, ref)
        # the same with RF input: quadrature pre-pass (edge rule applied as a post-pass over the chunk image) at both
        # precisions, and the generic pre-pass (fs != 4 fc)
        for extra in (dict(), dict(fs=25e6, fc=5.21e6)):
            cfg = small(t_start=t_start, n_samples=ns, **extra)
            ch = synth.random_channel(cfg, 2, seed=32, amplitude=6000)
            check_noise(torch_cuda, cfg, ch)


@pytest.mark.parametrize("precision,bound", [(2, 2e-5), (0, 1e-4), (1, 2e-4)])
def test_linearity_on_gpu(torch_cuda, precision, bound):
    """B(a + b) = B(a) + B(b): to fp32 rounding with the full scratch format; the compact formats round the
    difference term to fp16, which is linear only up to that rounding: within the
    1e-4 bar for the default format, at the documented format bound for the opt-in fast one (precision = 1)."""
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    cfg = small()
    a = synth.random_channel(cfg, 2, seed=1, amplitude=8000)
    b = synth.random_channel(cfg, 2, seed=2, amplitude=8000)
    with Plan(**rounded_kwargs(cfg), precision=precision) as plan:
        assert plan.info()["precision"] == (precision or 3)
        outs = [plan.beamform(torch.from_numpy(v).cuda()).cpu().numpy() for v in (a, b, a + b)]
    s = np.abs(outs[2]).max()
    assert np.abs(outs[2] - (outs[0] + outs[1])).max() <= bound * s


def test_host_entry_matches_device_entry(torch_cuda):
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    d = synth.LAMBDA_M / 2
    folded = dict(grid_xz=centred_grid(37, d, 53, 6e-3, d), grid_yz=centred_grid(29, 1.2 * d, 41, 6.5e-3, 0.8 * d),
                  row_tx_angles=tuple(np.radians([-6.0, 2.0, 6.0])), t0=None)
    for over in (dict(), folded):
        cfg = small(**over)
        ch = synth.random_channel(cfg, 3, seed=8, amplitude=6000)
        with Plan(**rounded_kwargs(cfg)) as plan:
            dev = plan.beamform(torch.from_numpy(ch).cuda()).cpu().numpy()
            host = plan.beamform_host(ch)
        np.testing.assert_array_equal(dev, host)


@pytest.mark.parametrize("n_frames,precision", [(2, 0), (1, 2), (3, 0), (5, 2)])
def test_volume_small(torch_cuda, n_frames, precision):
    """Full 3-D comparator against the oracle's point-outer DAS on a small shared-axial-grid case: batches of one or
    two frames take unpack_frame_kernel + das_volume_kernel (plane counts 15 / 19 leave a ragged plane group),
    larger ones the generic kernel; compact and full scratch entries."""
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    d = synth.LAMBDA_M / 2
    gx = centred_grid(19, d, 33, 6e-3, d, ref=0.0)
    gy = centred_grid(15, 1.3 * d, 33, 6e-3, d, ref=0.0)
    cfg = small(grid_xz=gx, grid_yz=gy, n_frames=n_frames, f_number=1.4)
    ch = synth.random_channel(cfg, n_frames, seed=41, amplitude=6000)
    kw = rounded_kwargs(cfg)
    assert_mask_margin(kw)
    p = oracle.OracleParams(**kw)
    xs = kw["grid_xz"][1] + kw["grid_xz"][2] * np.arange(gx[0])
    ys = kw["grid_yz"][1] + kw["grid_yz"][2] * np.arange(gy[0])
    zs = kw["grid_xz"][4] + kw["grid_xz"][5] * np.arange(gx[3])
    with Plan(**kw, build_volume=True, precision=precision) as plan:
        vol = plan.beamform_volume(torch.from_numpy(ch).cuda()).cpu().numpy()
    for f in range(n_frames):
        v_rc, v_cr = oracle.volume(p, ch[f], xs, ys, zs)
        assert rel_err(vol[f], v_rc + v_cr) <= TOL


@pytest.mark.parametrize("nx,ny,sym,f_number", [(18, 14, True, 0.0), (18, 14, True, 1.4), (19, 14, True, 0.0), (18, 14, False, 1.4)])
def test_volume_mirror_pairs(torch_cuda, nx, ny, sym, f_number):
    """Single-frame volumes on mirror pairs (das_volume_mirror_kernel): centred grids with an even plane count, an angle
    set symmetric about 0 (with a theta = 0 event) and equal start delays share the index / weight / phasor arithmetic
    between (plane y, theta) and (plane -y, -theta); an odd plane count or an asymmetric angle set keeps
    das_volume_kernel.  Plane counts off the 3-planes-per-thread grouping (9 and 7 lower-half planes)."""
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    d = synth.LAMBDA_M / 2
    gx = centred_grid(nx, d, 33, 6e-3, d, ref=0.0)
    gy = centred_grid(ny, 1.3 * d, 33, 6e-3, d, ref=0.0)
    row = np.radians([-7.0, -2.5, 0.0, 2.5, 7.0]) if sym else np.radians([-7.0, 1.0, 6.0])
    col = np.radians([-4.0, 4.0]) if sym else np.radians([-4.0, 8.0])
    cfg = small(grid_xz=gx, grid_yz=gy, n_frames=2, f_number=f_number, row_tx_angles=tuple(row), col_tx_angles=tuple(col),
                t0=None if sym else (0.2e-6, -0.1e-6, 0.05e-6, 0.3e-6, -0.25e-6))
    ch = synth.random_channel(cfg, 2, seed=43, amplitude=6000)
    kw = rounded_kwargs(cfg)
    assert_mask_margin(kw)
    p = oracle.OracleParams(**kw)
    xs = kw["grid_xz"][1] + kw["grid_xz"][2] * np.arange(gx[0])
    ys = kw["grid_yz"][1] + kw["grid_yz"][2] * np.arange(gy[0])
    zs = kw["grid_xz"][4] + kw["grid_xz"][5] * np.arange(gx[3])
    with Plan(**kw, build_volume=True, precision=2) as plan:
        vol = plan.beamform_volume(torch.from_numpy(ch).cuda()).cpu().numpy()
        assert plan.info()["volume_mirror_pairs"] == int(sym and nx % 2 == 0 and ny % 2 == 0)
    for f in range(2):
        v_rc, v_cr = oracle.volume(p, ch[f], xs, ys, zs)
        assert rel_err(vol[f], v_rc + v_cr) <= NOISE_TOL_FULL


def test_config1_full_frame(torch_cuda):
    cfg = synth.config(1)
    ch = synth.render(cfg)
    gpu, ref, info = run_pair(torch_cuda, cfg, ch)
    worst = assert_parity(gpu, ref)
    print("cfg1 kernel=%d worst rel err %.3e" % (info["kernel"], worst))
    gpu, ref, info = run_pair(torch_cuda, cfg, ch, plan_extra=dict(kernel=1))
    worst = assert_parity(gpu, ref)
    print("cfg1 kernel=%d worst rel err %.3e" % (info["kernel"], worst))


def test_config4_volume_sampled(torch_cuda):
    """Config 4: cfg 1's data as a 180 x 180 x 164 volume; compared on three full planes and a random 0.2 %
    voxel subset (the full fp64 volume takes minutes on the host)."""
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    cfg = synth.config(4)
    ch = synth.render(cfg)
    kw = rounded_kwargs(cfg)
    p = oracle.OracleParams(**kw)
    gx, gy = kw["grid_xz"], kw["grid_yz"]
    xs = gx[1] + gx[2] * np.arange(gx[0])
    ys = gy[1] + gy[2] * np.arange(gy[0])
    zs = gx[4] + gx[5] * np.arange(gx[3])
    with Plan(**kw, build_volume=True) as plan:
        vol = plan.beamform_volume(torch.from_numpy(ch).cuda()).cpu().numpy()[0]
        proj = plan.beamform(torch.from_numpy(ch).cuda()).cpu().numpy()[0]
    rng = np.random.default_rng(4)
    n = 10000
    idx = np.stack([rng.integers(0, gx[0], n), rng.integers(0, gy[0], n), rng.integers(0, gx[3], n)], axis=1)
    planes = [np.stack(np.meshgrid([90], np.arange(gy[0]), np.arange(gx[3]), indexing="ij"), -1).reshape(-1, 3),
              np.stack(np.meshgrid(np.arange(gx[0]), [37], np.arange(gx[3]), indexing="ij"), -1).reshape(-1, 3),
              np.stack(np.meshgrid(np.arange(gx[0]), np.arange(gy[0]), [100], indexing="ij"), -1).reshape(-1, 3)]
    idx = np.concatenate([idx] + planes)
    pts = np.stack([xs[idx[:, 0]], ys[idx[:, 1]], zs[idx[:, 2]]], axis=1)
    v_rc, v_cr = oracle.das_points(p, ch[0], pts)
    ref = v_rc + v_cr
    got = vol[idx[:, 0], idx[:, 1], idx[:, 2]]
    scale = np.abs(ref).max()
    assert np.abs(got - ref).max() <= TOL * scale
    assert np.abs(vol).max() <= 1.5 * scale * 3       # no garbage anywhere in the volume


@pytest.mark.parametrize("index", [2, 3])
def test_ensemble_full_size_sampled(torch_cuda, index):
    """Configs 2 and 3 at full size in the launch configuration bench.py times (300 frames, one call,
    max_frames = 300): a few frames of the moving scene are rendered on the host, tiled over the 300-frame
    device buffer exactly as bench.py does, and every distinct frame is compared with the oracle at three
    positions of the ensemble (first group, a middle group, the last frame)."""
    torch = torch_cuda
    import bench
    from paper_2511_21647_b200 import Plan
    cfg = synth.config(index)
    dev = torch.device("cuda", 0)
    channel, host, distinct = bench.make_ensemble(cfg, torch, dev)
    kw = rounded_kwargs(cfg)
    p = oracle.OracleParams(**kw)
    check = [0, 1, 2, 3, 149, 150, 298, 299]
    with Plan(**kw, max_frames=cfg.n_frames) as plan:
        out = plan.beamform(channel)
        torch.cuda.synchronize()
        info = plan.info()
        got = out[check].cpu().numpy()
    # pre-pass + two-group ring launch (+ combine when its tail was split) + one-group launch for the odd 25th group (+ combine)
    assert info["kernel"] == 2 and 2 <= info["launches_last_call"] <= 5
    del out, channel
    refs = {}
    worst = 0.0
    for row, fr in enumerate(check):
        d = fr % len(distinct)
        if d not in refs:
            refs[d] = oracle.beamform(p, host[d][None])[0]
        e = rel_err(got[row], refs[d])
        worst = max(worst, e)
        assert e <= TOL, "cfg %d frame %d: %.3e" % (index, fr, e)
    print("PARITY cfg%d full size worst %.3e over frames %s" % (index, worst, check))


def test_fallback_to_generic_kernel_when_the_ring_does_not_cover_the_shape(torch_cuda):
    """More than 256 receive elements per aperture: kernel = auto must fall back to the generic gather kernel
    (and kernel = 2 must refuse), results still within tolerance."""
    from paper_2511_21647_b200 import Plan, UlmRcaError
    d = synth.LAMBDA_M / 2
    cfg = small(n_rows=6, n_cols=260, pitch=0.1e-3, n_frames=2, row_tx_angles=tuple(np.radians([-3.0, 2.0])),
                col_tx_angles=tuple(np.radians([4.0])), t0=(0.1e-6, -0.1e-6, 0.2e-6),
                grid_xz=centred_grid(21, d, 17, 6e-3, d), grid_yz=centred_grid(9, d, 13, 6e-3, d))
    ch = synth.random_channel(cfg, 2, seed=3, amplitude=6000)
    gpu, ref, info = check_noise(torch_cuda, cfg, ch)
    assert info["kernel"] == 1
    with pytest.raises(UlmRcaError) as ei:
        Plan(**rounded_kwargs(cfg), kernel=2)
    assert ei.value.status == 4


def test_many_frames_cross_group_boundaries(torch_cuda):
    """25 frames = two full 12-frame groups + 1: every frame, including the lone one of the last group (the first two
    groups go through the two-group work items, the third through a launch of one-group items)."""
    cfg = small(n_frames=25)
    ch = synth.random_channel(cfg, 25, seed=29, amplitude=3000)
    ch = (ch.astype(np.int32) + synth.random_channel(cfg, 25, seed=30, amplitude=3000)).astype(np.int16)
    gpu, ref, info = check_noise(torch_cuda, cfg, ch, plan_extra=dict(max_frames=25))
    assert 3 <= info["launches_last_call"] <= 5     # pre-pass, two ring launches, a combine kernel for each split one


@pytest.mark.parametrize("compound,f_number,precision,frames", [
    (1, 0.0, 0, 24), (1, 1.3, 0, 37), (0, 0.0, 0, 26), (0, 1.3, 1, 30), (1, 0.0, 1, 49), (1, 1.3, 2, 30)])
def test_two_group_work_items(torch_cuda, compound, f_number, precision, frames):
    """Calls of more than 12 frames with compact entries run the ring kernel on work items of TWO frame groups (24
    frames, tiles of 2 rows); an odd last group goes through a launch of one-group items.  Every variant of that kernel
    (apodisation on / off, one- and two-term weight, compounded / per-angle) against the oracle on every frame; the
    full-entry plan (precision 2) keeps the one-group items and must agree as well."""
    cfg = small(n_frames=frames, compound=compound, f_number=f_number)
    ch = synth.random_channel(cfg, frames, seed=70 + frames, amplitude=5000)
    extra = dict(max_frames=frames)
    if precision:
        extra["precision"] = precision
    gpu, ref, info = check_noise(torch_cuda, cfg, ch, plan_extra=extra)
    assert info["kernel"] == 2 and info["precision"] == (precision or 3)
    assert (info["window_two_groups"] > 0 and info["stages_two_groups"] >= 3) == (info["precision"] != 2)


def test_tail_split_of_the_last_round(torch_cuda):
    """More work items than SMs with a partially filled last round: those items are cut into slices of the receive
    elements whose partial sums a second kernel adds in slice order (compounded and per-angle).  48 frames = two pairs of
    frame groups, so the call is one launch of two-group work items (tiles of 384 positions x 2 rows)."""
    torch = torch_cuda
    n_sms = torch.cuda.get_device_properties(0).multi_processor_count
    d = synth.LAMBDA_M / 2
    g = centred_grid(200, 0.25 * d, 200, 6e-3, 0.5 * d)
    frames = 48
    for compound in (1, 0):
        cfg = small(grid_xz=g, grid_yz=g, n_frames=frames, compound=compound)
        tiles2 = -(-(200 * 100) // 384)
        n_tx = len(cfg.row_tx_angles) + len(cfg.col_tx_angles)
        items = 2 * tiles2 * (2 if compound else n_tx)
        ch = synth.random_channel(cfg, frames, seed=55 + compound, amplitude=6000)
        gpu, ref, info = check_noise(torch_cuda, cfg, ch, plan_extra=dict(max_frames=frames))
        assert info["kernel"] == 2
        if compound:
            assert info["tiles_xz"] == -(-(200 * 50) // 384)
        if n_sms == 148:
            assert items > n_sms and items % n_sms != 0
            assert info["launches_last_call"] == 3, info       # pre-pass, ring kernel, combine kernel


SWEEP = [
    # n_rows, n_cols, n_lat_xz, n_ax_xz, n_lat_yz, n_ax_yz, n_row_tx, n_col_tx, frames, dz scale, f_number
    (9, 40, 5, 3, 7, 4, 1, 2, 1, 1.0, 0.0),
    (33, 17, 97, 50, 61, 37, 2, 1, 5, 0.7, 0.0),
    (16, 48, 200, 9, 150, 21, 3, 2, 13, 1.3, 1.2),
    (40, 40, 31, 130, 31, 130, 5, 5, 4, 0.5, 0.0),
    (12, 64, 385, 4, 383, 5, 2, 2, 3, 1.0, 2.1),
]


@pytest.mark.parametrize("shape", SWEEP)
def test_shape_sweep_ring_kernel(torch_cuda, shape):
    """Odd shapes through the ring kernel: fewer positions than one tile, one-row images, tiles that span many
    strips, wide images, many frames, f-number masks -- window planning and the ragged tails."""
    n_rows, n_cols, nlx, nax, nly, nay, kr, kc, nf, dzs, fnum = shape
    d = synth.LAMBDA_M / 2
    rng = np.random.default_rng(sum(shape[:9]))
    cfg = synth.config(0).with_(
        n_rows=n_rows, n_cols=n_cols, pitch=0.25e-3, n_samples=900,
        row_tx_angles=tuple(np.radians(rng.uniform(-9, 9, kr))), col_tx_angles=tuple(np.radians(rng.uniform(-9, 9, kc))),
        grid_xz=centred_grid(nlx, 0.6 * d, nax, 5e-3, dzs * d, ref=0.2e-3),
        grid_yz=centred_grid(nly, 0.5 * d, nay, 5.5e-3, dzs * d, ref=-0.1e-3),
        n_frames=nf, t_start=0.4e-6, t0=tuple(rng.uniform(-0.2e-6, 0.2e-6, kr + kc)), f_number=fnum)
    ch = synth.random_channel(cfg, nf, seed=int(rng.integers(1 << 30)), amplitude=4000)
    # full entries: nothing but fp32 rounding, so a planning / indexing mistake anywhere shows up at once
    gpu, ref, info = run_pair(torch_cuda, cfg, ch, plan_extra=dict(max_frames=nf, precision=2))
    assert info["kernel"] == 2 and info["precision"] == 2
    assert_parity(gpu, ref, tol=2e-5)
    # the default entries (compact, two-term weight) on the same noise-only data: the north-star bar
    gpu, ref, info = run_pair(torch_cuda, cfg, ch, plan_extra=dict(max_frames=nf))
    assert info["kernel"] == 2 and info["precision"] == 3
    assert_parity(gpu, ref, tol=TOL)


def _random_case(rng):
    """One random small configuration: array, angle sets (symmetric ones fold), grids, frames, apodisation, mode."""
    d = synth.LAMBDA_M / 2
    n_rows, n_cols = int(rng.integers(4, 70)), int(rng.integers(4, 70))
    kr, kc = int(rng.integers(0, 6)), int(rng.integers(0, 6))
    if kr + kc == 0:
        kr = 1
    sym = rng.random() < 0.5

    def angles(k):
        if sym:
            return tuple(np.radians(np.linspace(-1, 1, k) * rng.uniform(1, 10) if k > 1 else np.zeros(k)))
        return tuple(np.radians(rng.uniform(-10, 10, k)))

    volume = rng.random() < 0.25
    nf = int(rng.choice([1, 2, 3, 5]) if volume else rng.choice([1, 2, 3, 4, 5, 12, 13, 25, 30]))
    nlx, nly, nax = int(rng.integers(1, 120)), int(rng.integers(1, 120)), int(rng.integers(1, 90))
    nay = int(rng.integers(1, 90))
    if volume:
        nlx, nly, nax = min(nlx, 24), min(nly, 24), min(nax, 30)
        nay = nax
    dz, z0 = d * rng.uniform(0.4, 1.5), rng.uniform(3e-3, 8e-3)
    ref_x, ref_y = (0.0, 0.0) if sym else (rng.uniform(-1e-3, 1e-3), rng.uniform(-1e-3, 1e-3))
    t0 = None if (sym or rng.random() < 0.5) else tuple(rng.uniform(-0.2e-6, 0.2e-6, kr + kc))
    # sampling rate / filter: quadrature pre-pass (fs = 4 fc), generic (fs = 5 fc, other tap counts), analytic (fs = 8 fc)
    fs = float(rng.choice([20e6, 20e6, 25e6, 40e6, 40e6]))
    cfg = synth.config(0).with_(
        fs=fs, demod_taps=int(rng.choice([0, 0, 0, 9, 25])), input_kind=int(rng.random() < 0.15),
        n_rows=n_rows, n_cols=n_cols, pitch=float(rng.uniform(0.15e-3, 0.35e-3)),
        n_samples=int(rng.integers(300, 1400) * (2 if fs == 40e6 else 1)),
        row_tx_angles=angles(kr), col_tx_angles=angles(kc),
        grid_xz=centred_grid(nlx, d * rng.uniform(0.3, 1.2), nax, z0, dz, ref=ref_y),
        grid_yz=centred_grid(nly, d * rng.uniform(0.3, 1.2), nay, z0, dz, ref=ref_x),
        n_frames=nf, t_start=float(rng.uniform(0, 1e-6)), t0=t0, f_number=float(rng.choice([0.0, 0.0, 1.0, 1.7])),
        compound=int(rng.random() < 0.7))
    extra = dict(kernel=int(rng.choice([0, 0, 1])), max_frames=int(rng.choice([nf, max(1, nf // 2), 32])),
                 build_volume=bool(volume), precision=2)
    return cfg, nf, extra


def test_two_group_items_on_random_shapes(torch_cuda):
    """The work items of two frame groups against the one-group items of the SAME compact scratch format on seeded
    random configurations (tile and window planning with 2-row strips, odd last groups, per-angle output, f-number
    masks, all three pre-pass kernels): a call of 13..45 frames (two-group items, + a one-group launch for an odd last
    group) must reproduce the same frames beamformed 12 at a time (one-group items; frames keep their 4-frame chunk
    mates inside full chunks).  What may differ: the order of the fp32 additions (split tail items add their element
    slices in slice order, and which items are split depends on the item count) and, in a partly filled last chunk, the
    foreign low mantissa byte of the fp24 mid values (include/ulm_rca.h; bounded at 5e-5 of the image maximum by
    test_plan_reuse_and_determinism): measured <= 2.3e-5 over 660 seeded shapes, tested at 5e-5 -- three orders of
    magnitude below what a planning or indexing mistake gives."""
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    done = 0
    for it in range(60):
        rng = np.random.default_rng(9100 + it)
        cfg, _, extra = _random_case(rng)
        if cfg.input_kind == 1:
            continue                          # IQ input is staged as full entries: one-group items only
        nf = int(rng.integers(13, 46))
        cfg = cfg.with_(n_frames=nf)
        ch = synth.random_channel(cfg, nf, seed=int(rng.integers(1 << 30)), amplitude=5000)
        kw = rounded_kwargs(cfg)
        with Plan(**kw, max_frames=nf, precision=int(rng.choice([1, 3])), kernel=2) as plan:
            d_ch = torch.from_numpy(ch).cuda()
            whole = plan.beamform(d_ch).cpu().numpy()
            launches = plan.info()["launches_last_call"]
            parts = np.concatenate([plan.beamform(d_ch[f0:f0 + 12]).cpu().numpy() for f0 in range(0, nf, 12)])
        scale = np.abs(parts).max()
        assert scale > 0 and launches >= 2
        err = np.abs(whole - parts).max() / scale
        assert err <= 5e-5, (it, nf, err, cfg)
        done += 1
    assert done >= 40


@pytest.mark.parametrize("block", range(4))
def test_random_shapes(torch_cuda, block):
    """Seeded random configurations (40 per block) against the oracle with full-precision entries, where only fp32
    rounding separates the two (2e-5 on white noise; 4e-5 for unfiltered white IQ input): array
    sizes, 0..5 angles per aperture (symmetric sets fold), one-pixel to multi-tile grids, records that end inside the
    image, 1..30 frames in batches, f-number masks, per-angle output, fs = 4 / 5 / 8 fc and three tap counts (all three
    pre-pass kernels), RF and IQ input, both DAS kernels, and the volume path on a quarter of the cases."""
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    for it in range(40):
        rng = np.random.default_rng(7000 + 40 * block + it)
        cfg, nf, extra = _random_case(rng)
        ch = synth.random_channel(cfg, nf, seed=int(rng.integers(1 << 30)), amplitude=5000)
        kw = rounded_kwargs(cfg)
        while mask_margin(kw) < 1e-6:       # a pair on the mask edge (to fp32 rounding): move the f-number off it
            cfg = cfg.with_(f_number=cfg.f_number * 1.0001)
            kw = rounded_kwargs(cfg)
        p = oracle.OracleParams(**kw)
        with Plan(**kw, **extra) as plan:
            d_ch = torch.from_numpy(ch).cuda()
            out = plan.beamform(d_ch).cpu().numpy()
            vol = plan.beamform_volume(d_ch).cpu().numpy() if extra["build_volume"] else None
        err = rel_err(out, oracle.beamform(p, ch))
        if vol is not None:
            gx, gy = kw["grid_xz"], kw["grid_yz"]
            xs, ys = gx[1] + gx[2] * np.arange(gx[0]), gy[1] + gy[2] * np.arange(gy[0])
            zs = gx[4] + gx[5] * np.arange(gx[3])
            for f in range(nf):
                v_rc, v_cr = oracle.volume(p, ch[f], xs, ys, zs)
                err = max(err, rel_err(vol[f], v_rc + v_cr))
        assert err <= (2 * NOISE_TOL_FULL if cfg.input_kind == 1 else NOISE_TOL_FULL), (block, it, err, cfg)

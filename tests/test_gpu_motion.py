"""GPU parity of the Fourier-domain NCC motion estimation (ulm_rca_motion_estimate) against
oracle/motion.py through the C-ABI.

Bars: the integer peak location is an index and must agree exactly; the sub-pixel shifts agree
within 1e-3 pixel and the NCC peak within 1e-4 (fp32 transforms against fp64: errors of ~1e-6 of the peak are amplified
by the inverse curvature of the parabola); the per-frame motion within 1e-3 of a pixel size."""
import numpy as np
import pytest

import oracle
import synth
from helpers import rounded_kwargs
from oracle import motion
from synth import centred_grid

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2511_21647_b200 import build
    build.build()
    return torch


def cfg_of(nlx, nzx, nly, nzy, kr=2, kc=1, **kw):
    d = synth.LAMBDA_M / 2
    ang = np.radians([-5.0, 3.0, 7.0, -2.0])
    base = dict(n_rows=24, n_cols=20, pitch=0.3e-3, n_samples=900, compound=0, n_frames=1,
                row_tx_angles=tuple(ang[:kr]), col_tx_angles=tuple(ang[:kc]),
                grid_xz=centred_grid(nlx, 1.1 * d, nzx, 6e-3, 0.5 * d), grid_yz=centred_grid(nly, 1.3 * d, nzy, 6e-3, 0.7 * d))
    base.update(kw)
    return synth.config(0).with_(**base)


def shapes_of(cfg):
    return [(cfg.grid_xz[0], cfg.grid_xz[3])] * len(cfg.row_tx_angles) + [(cfg.grid_yz[0], cfg.grid_yz[3])] * len(cfg.col_tx_angles)


def check(torch, cfg, slices, ref_frame=0, max_frames=None):
    from paper_2511_21647_b200 import Plan
    kw = rounded_kwargs(cfg)
    per_ref, mot_ref = motion.estimate(oracle.OracleParams(**kw), slices.astype(np.complex128), ref_frame)
    with Plan(**kw, motion_frames=max_frames or slices.shape[0]) as plan:
        mot, per = plan.motion_estimate(torch.from_numpy(slices).cuda(), ref_frame)
        torch.cuda.synchronize()
        assert plan.info()["launches_last_call"] == 6
        mot, per = mot.cpu().numpy(), per.cpu().numpy()
    e_shift = np.abs(per[:, :, :2] - per_ref[:, :, :2]).max()
    e_ncc = np.abs(per[:, :, 2] - per_ref[:, :, 2]).max()
    px = min(abs(kw["grid_xz"][2]), abs(kw["grid_yz"][2]), kw["grid_xz"][5], kw["grid_yz"][5])
    e_mot = np.abs(mot[:, :3] - mot_ref[:, :3]).max() / px
    print("MOTION shift err %.2e px, ncc err %.2e, motion err %.2e px; shifts up to %.2f px, ncc >= %.3f" %
          (e_shift, e_ncc, e_mot, np.abs(per_ref[:, :, :2]).max(), per_ref[:, :, 2].min()))
    assert np.array_equal(np.round(per[:, :, :2] - (per[:, :, :2] - np.round(per_ref[:, :, :2]))), np.round(per_ref[:, :, :2]))
    assert e_shift <= 1e-3 and e_ncc <= 1e-4 and e_mot <= 1e-3
    return per_ref, mot_ref


@pytest.mark.parametrize("shape", [(37, 53, 29, 41), (64, 32, 33, 100), (180, 164, 180, 164)])
def test_known_motion_is_recovered_and_matches_the_oracle(torch_cuda, shape):
    cfg = cfg_of(*shape)
    shifts = [(0.0, 0.0), (0.4, -0.3), (1.5, 0.75), (-2.2, 1.9), (3.0, -4.0), (0.05, 0.5)]
    s = synth.moving_speckle(len(shifts), shapes_of(cfg), shifts, seed=sum(shape))
    per_ref, _ = check(torch_cuda, cfg, s)
    # and the estimator itself finds the programmed motion (speckle decorrelation, noise and the content that enters /
    # leaves at the image edges bias it: a fraction of a pixel on the full-size slices, more on the small ones)
    worst = np.abs(per_ref[:, :, :2] - np.array(shifts)[:, None, :]).max()
    print("MOTION estimator vs programmed motion: worst %.3f px" % worst)
    assert worst < (0.25 if shape[0] >= 180 else 1.0)


def test_reference_frame_batches_and_single_aperture(torch_cuda):
    cfg = cfg_of(40, 48, 36, 44, kr=0, kc=3)
    shifts = [(0.5 * f, -0.25 * f) for f in range(5)]
    s = synth.moving_speckle(5, shapes_of(cfg), shifts, seed=9)
    per_ref, mot_ref = check(torch_cuda, cfg, s, ref_frame=3, max_frames=8)
    assert np.abs(per_ref[3, :, :2]).max() < 1e-9 and abs(mot_ref[3, 3] - 1.0) < 1e-9
    assert np.all(mot_ref[:, 0] == 0.0)                    # no row-tx events: no x motion


def test_fine_grid_size_and_bad_arguments(torch_cuda):
    """cfg 3's slice size (360 x 328 -> 512 x 512 transforms); argument checks."""
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan, UlmRcaError
    cfg = cfg_of(360, 328, 360, 328, kr=1, kc=1)
    shifts = [(0.0, 0.0), (2.3, -1.6)]
    s = synth.moving_speckle(2, shapes_of(cfg), shifts, seed=4, correlation_px=4.0)
    check(torch, cfg, s)
    with Plan(**rounded_kwargs(cfg), motion_frames=2) as plan:
        d = torch.from_numpy(s).cuda()
        with pytest.raises(UlmRcaError):
            plan.motion_estimate(torch.cat([d, d]), 0)          # more frames than motion_frames
        with pytest.raises(UlmRcaError):
            plan.motion_estimate(d, 2)                           # reference outside the call
    with Plan(**rounded_kwargs(cfg)) as plan:
        with pytest.raises(ValueError):
            plan.motion_estimate(torch.from_numpy(s).cuda(), 0)
    big = cfg_of(600, 64, 64, 64)
    with pytest.raises(UlmRcaError) as ei:
        Plan(**rounded_kwargs(big), motion_frames=2)
    assert ei.value.status == 4


def test_config2_ensemble_size_sampled(torch_cuda):
    """The launch configuration bench.py times: 300 frames x 22 slices of 180 x 164 px in one call; frames 1, 150 and 299
    are checked against the oracle for every event (the ensemble is a few distinct frames tiled, as in bench.py)."""
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    cfg = synth.config(2).with_(compound=0)
    kw = rounded_kwargs(cfg)
    shapes = shapes_of(cfg)
    shifts = [(0.0, 0.0), (0.8, -0.6), (-1.4, 0.35), (2.6, 1.2)]
    distinct = synth.moving_speckle(4, shapes, shifts, seed=2)
    idx = torch.arange(300, device="cuda") % 4
    d = torch.from_numpy(distinct).cuda()[idx].contiguous()
    with Plan(**kw, motion_frames=300) as plan:
        mot, per = plan.motion_estimate(d, 0)
        torch.cuda.synchronize()
        print("MOTION cfg2 size: %.3f ms per 300-frame ensemble" % plan.motion_timing())
        mot, per = mot.cpu().numpy(), per.cpu().numpy()
    per_ref, mot_ref = motion.estimate(oracle.OracleParams(**kw), distinct.astype(np.complex128), 0)
    for f in (1, 150, 299):
        assert np.abs(per[f, :, :2] - per_ref[f % 4, :, :2]).max() <= 1e-3
        assert np.abs(per[f, :, 2] - per_ref[f % 4, :, 2]).max() <= 1e-4
        assert np.abs(mot[f, :3] - mot_ref[f % 4, :3]).max() <= 1e-3 * kw["grid_xz"][5]

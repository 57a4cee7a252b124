"""GPU parity of Stage 2 + compounding + P-block sum-projection (ulm_rca_stage2_project)
against oracle/stage2.py, element by element, through the C-ABI.  Bar: max|gpu - oracle| <= 1e-4 max|oracle| per frame."""
import numpy as np
import pytest

import oracle
import synth
from helpers import rel_err, rounded_kwargs
from oracle import stage2
from synth import centred_grid

pytestmark = pytest.mark.gpu
TOL = 1e-4


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2511_21647_b200 import build
    build.build()
    return torch


def base_cfg(**kw):
    d = synth.LAMBDA_M / 2
    base = dict(n_rows=24, n_cols=20, pitch=0.3e-3, n_samples=900, compound=0, n_frames=2, t_start=0.4e-6,
                row_tx_angles=tuple(np.radians([-7.0, 0.0, 1.0, 6.0])), col_tx_angles=tuple(np.radians([-4.0, 8.0, 3.0])),
                grid_xz=centred_grid(37, d, 53, 6e-3, d, ref=0.4e-3), grid_yz=centred_grid(45, 1.2 * d, 53, 6e-3, d, ref=-0.3e-3),
                t0=(0.2e-6, -0.1e-6, 0.05e-6, 0.0, 0.3e-6, -0.25e-6, 0.1e-6))
    base.update(kw)
    return synth.config(0).with_(**base)


def slices_shape(cfg, n_frames):
    return (n_frames, len(cfg.row_tx_angles) * cfg.grid_xz[0] * cfg.grid_xz[3] + len(cfg.col_tx_angles) * cfg.grid_yz[0] * cfg.grid_yz[3])


def check(torch, cfg, block, n_frames=None, seed=1, plan_extra=None):
    """Seeded random complex slices through ulm_rca_stage2_project and through the oracle."""
    from paper_2511_21647_b200 import Plan
    n_frames = n_frames or cfg.n_frames
    kw = rounded_kwargs(cfg)
    s = synth.random_complex(slices_shape(cfg, n_frames), seed, amplitude=100.0)
    ref = stage2.stage2_planes(oracle.OracleParams(**kw), s.astype(np.complex128), block)
    with Plan(**kw, stage2_block=block, **(plan_extra or {})) as plan:
        out = plan.stage2_project(torch.from_numpy(s).cuda())
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert plan.n_planes_xz == -(-cfg.grid_yz[0] // block) and plan.n_planes_yz == -(-cfg.grid_xz[0] // block)
        assert plan.info()["launches_last_call"] == 2 * -(-n_frames // (plan_extra or {}).get("max_frames", 32))
    assert got.shape == ref.shape
    worst = max(rel_err(got[f], ref[f]) for f in range(n_frames))
    print("STAGE2 PARITY block %d worst %.3e over %d frame(s)" % (block, worst, n_frames))
    assert worst <= TOL
    return worst


@pytest.mark.parametrize("block", [8, 3, 1, 64])
def test_block_sizes(torch_cuda, block):
    """P = 8, a block that leaves ragged last groups, single columns, a block wider than the grid."""
    check(torch_cuda, base_cfg(), block)


@pytest.mark.parametrize("case", ["neg_dlat", "one_aperture_rc", "one_aperture_cr", "wide", "deep", "tiny", "steep", "frames"])
def test_shapes(torch_cuda, case):
    d = synth.LAMBDA_M / 2
    extra = None
    if case == "neg_dlat":
        g = base_cfg().grid_xz
        cfg = base_cfg(grid_xz=(g[0], g[1] + (g[0] - 1) * g[2], -g[2]) + g[3:])
    elif case == "one_aperture_rc":
        cfg = base_cfg(col_tx_angles=(), t0=(0.2e-6, -0.1e-6, 0.05e-6, 0.0))
    elif case == "one_aperture_cr":
        cfg = base_cfg(row_tx_angles=(), t0=(0.3e-6, -0.25e-6, 0.1e-6))
    elif case == "wide":        # several lateral tiles of 32 with ragged tails, more than 8 groups (two group blocks)
        cfg = base_cfg(grid_xz=centred_grid(101, 0.5 * d, 30, 6e-3, d, ref=0.0), grid_yz=centred_grid(75, 0.5 * d, 30, 6e-3, d, ref=0.2e-3))
    elif case == "deep":        # several depth tiles of 24 with a ragged tail, odd n_z (scalar stores)
        cfg = base_cfg(grid_xz=centred_grid(9, d, 131, 6e-3, 0.5 * d, ref=0.0), grid_yz=centred_grid(12, d, 131, 6e-3, 0.5 * d, ref=0.0))
    elif case == "tiny":        # one pixel column, two depths
        cfg = base_cfg(grid_xz=centred_grid(1, d, 2, 6e-3, d, ref=0.0), grid_yz=centred_grid(3, d, 2, 6e-3, d, ref=0.0))
    elif case == "steep":       # 15 degrees, fine depth step: shifts of many pixels, 4 .. 6 taps per group
        cfg = base_cfg(row_tx_angles=tuple(np.radians([-15.0, 15.0])), col_tx_angles=tuple(np.radians([12.0])), t0=None,
                       grid_xz=centred_grid(40, d, 80, 6e-3, 0.25 * d, ref=0.0), grid_yz=centred_grid(40, d, 80, 6e-3, 0.25 * d, ref=0.0))
    else:                        # more frames than max_frames: batches
        cfg = base_cfg(n_frames=7)
        extra = dict(max_frames=3)
    check(torch_cuda, cfg, 8, plan_extra=extra)


def test_unsupported_shift_range_is_refused(torch_cuda):
    from paper_2511_21647_b200 import Plan, UlmRcaError
    d = synth.LAMBDA_M / 2
    cfg = base_cfg(row_tx_angles=tuple(np.radians([-40.0, 40.0])), col_tx_angles=(), t0=None,
                   grid_xz=centred_grid(40, d, 80, 6e-3, 0.1 * d), grid_yz=centred_grid(200, d, 80, 6e-3, 0.1 * d))
    with pytest.raises(UlmRcaError) as ei:
        Plan(**rounded_kwargs(cfg), stage2_block=8)
    assert ei.value.status == 4
    with Plan(**rounded_kwargs(base_cfg())) as plan:
        with pytest.raises(ValueError):
            plan.stage2_project(torch_cuda.zeros((1, 4), dtype=torch_cuda.complex64, device="cuda"))


def test_chain_stage1_stage2_on_echo_data(torch_cuda):
    """Channel data -> per-event slices (ulm_rca_beamform, compound = 0) -> projected planes, both on the GPU, against
    the oracle chain on the same channel data (config 0's scene, 3 + 3 angles)."""
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    cfg = synth.config(0).with_(compound=0)
    ch = synth.render(cfg)
    kw = rounded_kwargs(cfg)
    p = oracle.OracleParams(**kw)
    ref = stage2.stage2_planes(p, oracle.beamform(p, ch), 8)
    with Plan(**kw, stage2_block=8) as plan:
        s = plan.beamform(torch.from_numpy(ch).cuda())
        got = plan.stage2_project(s).cpu().numpy()
    worst = max(rel_err(got[f], ref[f]) for f in range(ref.shape[0]))
    print("STAGE2 PARITY chain cfg0 worst %.3e" % worst)
    assert worst <= TOL


def test_config1_full_size_and_config2_sampled(torch_cuda):
    """cfg 1 (180 x 180 x 164 voxels, 11 + 11 events, P = 8 -> 23 + 23 planes) element by element; cfg 2 in the launch
    configuration bench.py times (300 frames, one call): frames 0, 151 and 299 against the oracle."""
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    cfg = synth.config(1).with_(compound=0)
    kw = rounded_kwargs(cfg)
    p = oracle.OracleParams(**kw)
    n_frames = 300
    distinct = synth.random_complex(slices_shape(cfg, 3), 21, amplitude=50.0)
    idx = torch.arange(n_frames, device="cuda") % 3
    slices = torch.from_numpy(distinct).cuda()[idx].contiguous()
    with Plan(**kw, stage2_block=8, max_frames=n_frames) as plan:
        out = plan.stage2_project(slices)
        torch.cuda.synchronize()
        got = out[[0, 151, 299]].cpu().numpy()
        assert plan.n_planes_xz == 23 and plan.n_planes_yz == 23
    del out, slices
    refs = stage2.stage2_planes(p, distinct.astype(np.complex128), 8)
    for row, fr in enumerate([0, 151, 299]):
        e = rel_err(got[row], refs[fr % 3])
        print("STAGE2 PARITY cfg2 frame %d: %.3e" % (fr, e))
        assert e <= TOL

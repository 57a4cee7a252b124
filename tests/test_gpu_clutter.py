"""GPU parity of the eigen-based clutter filter (ulm_rca_clutter_filter) against oracle/clutter.py through
the C-ABI.

Tolerances: the covariance is a linear map of the slices formed from bf16 (hi, lo) splits with the
lo x lo term dropped and fp32 accumulation: |C_gpu - C_oracle| <= 1e-4 max|C|.  The eigenvalues inherit that bound
(|d lambda| <= ||dC||).  The filtered slices are compared relative to the INPUT scale, max|gpu - oracle| <= 1e-4 max|X|:
the output is the small difference X - X P_c of quantities of the input's size, and a perturbation dC of the covariance
turns the clutter subspace by ~||dC|| / gap, which leaks that fraction of the (input-sized) clutter into the result; the
test data have tissue 30 dB above blood and an eigen-gap of > 100 at the chosen rank, as the filter assumes."""
import numpy as np
import pytest

import oracle
import synth
from helpers import rounded_kwargs
from oracle import clutter
from synth import centred_grid

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2511_21647_b200 import build
    build.build()
    return torch


def small_cfg(**kw):
    d = synth.LAMBDA_M / 2
    base = dict(n_rows=24, n_cols=20, pitch=0.3e-3, n_samples=900, compound=0, n_frames=1,
                row_tx_angles=tuple(np.radians([-7.0, 0.0, 6.0])), col_tx_angles=tuple(np.radians([-4.0, 8.0])),
                grid_xz=centred_grid(37, d, 53, 6e-3, d), grid_yz=centred_grid(29, d, 41, 6e-3, d))
    base.update(kw)
    return synth.config(0).with_(**base)


def n_pix_list(cfg):
    return [cfg.grid_xz[0] * cfg.grid_xz[3]] * len(cfg.row_tx_angles) + [cfg.grid_yz[0] * cfg.grid_yz[3]] * len(cfg.col_tx_angles)


def run(torch, cfg, x, rank, n_t_max=None, in_place=False):
    from paper_2511_21647_b200 import Plan
    with Plan(**rounded_kwargs(cfg), clutter_frames=n_t_max or x.shape[0]) as plan:
        d_x = torch.from_numpy(x).cuda()
        out, lam, cov = plan.clutter_filter(d_x, rank, out=d_x if in_place else None, want_eigenvalues=True, want_covariance=True)
        torch.cuda.synchronize()
        assert plan.info()["launches_last_call"] == 5
        return out.cpu().numpy(), lam.cpu().numpy(), cov.cpu().numpy()


def check(torch, cfg, x, rank, **kw):
    p = oracle.OracleParams(**rounded_kwargs(cfg))
    ref, lam_ref = clutter.clutter_filter(p, x.astype(np.complex128), rank)
    got, lam, cov = run(torch, cfg, x, rank, **kw)
    scale = np.abs(x).max()
    for e, (off, n) in enumerate(clutter.event_blocks(p)):
        c_ref = clutter.covariance(x[:, off:off + n].astype(np.complex128))
        e_cov = np.abs(cov[e] - c_ref).max() / np.abs(c_ref).max()
        e_lam = np.abs(lam[e][:rank + 2] - lam_ref[e][:rank + 2]).max() / lam_ref[e][0]
        e_out = np.abs(got[:, off:off + n] - ref[:, off:off + n]).max() / scale
        gap = lam_ref[e][rank - 1] / lam_ref[e][rank] if rank > 0 else float("inf")
        print("CLUTTER event %d: cov %.2e  eigenvalues %.2e  filtered %.2e (of max|X|)  gap lambda_r/lambda_r+1 = %.1f" % (e, e_cov, e_lam, e_out, gap))
        assert e_cov <= 1e-4 and e_lam <= 1e-4 and e_out <= 1e-4
        assert np.abs(cov[e] - cov[e].conj().T).max() <= 1e-6 * np.abs(c_ref).max()       # Hermitian by construction
    return got, ref


@pytest.mark.parametrize("n_t,rank", [(40, 3), (64, 3), (100, 5), (33, 1)])
def test_small_ensembles(torch_cuda, n_t, rank):
    """Two apertures with different slice sizes (1961 / 1189 px: ragged k-blocks of 64), n_t off the 64 / 128 tile sizes."""
    cfg = small_cfg()
    x = synth.clutter_ensemble(n_t, n_pix_list(cfg), seed=n_t, tissue_rank=rank)
    check(torch_cuda, cfg, x, rank)


def test_rank_zero_is_the_identity_and_in_place_works(torch_cuda):
    cfg = small_cfg()
    x = synth.clutter_ensemble(48, n_pix_list(cfg), seed=2, tissue_rank=2)
    got, _, _ = run(torch_cuda, cfg, x, 0)
    np.testing.assert_array_equal(got, x)
    a, _, _ = run(torch_cuda, cfg, x, 2)
    b, _, _ = run(torch_cuda, cfg, x, 2, in_place=True)
    np.testing.assert_array_equal(a, b)


def test_rank_deficient_covariance_is_deflated_not_normalised_into_noise(torch_cuda):
    """An ensemble of repeated frames (here 3 distinct frames, so C has rank 3 < the 32 iteration vectors): the
    surplus vectors have nothing to converge to and are deflated to zero; asking for the 3 (or more) clutter components
    removes everything, exactly as the oracle does.  (Found by chaining the stages on bench.py's tiled ensemble.)"""
    cfg = small_cfg()
    base = synth.clutter_ensemble(3, n_pix_list(cfg), seed=8, tissue_rank=2)
    x = np.ascontiguousarray(base[np.arange(48) % 3])
    p = oracle.OracleParams(**rounded_kwargs(cfg))
    for rank in (3, 5):
        got, lam, _ = run(torch_cuda, cfg, x, rank)
        ref, lam_ref = clutter.clutter_filter(p, x.astype(np.complex128), rank)
        assert np.isfinite(got).all() and np.isfinite(lam).all()
        assert np.abs(got - ref).max() <= 1e-4 * np.abs(x).max()
        assert np.abs(lam[:, :5] - lam_ref[:, :5]).max() <= 1e-4 * lam_ref[:, 0].max()
    got, _, _ = run(torch_cuda, cfg, x, 1)                    # one component of three: still well defined
    ref, _ = clutter.clutter_filter(p, x.astype(np.complex128), 1)
    assert np.abs(got - ref).max() <= 1e-4 * np.abs(x).max()


def test_smaller_call_on_a_larger_plan_and_bad_arguments(torch_cuda):
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan, UlmRcaError
    cfg = small_cfg()
    x = synth.clutter_ensemble(72, n_pix_list(cfg), seed=5, tissue_rank=3)
    check(torch, cfg, x, 3, n_t_max=130)
    with Plan(**rounded_kwargs(cfg), clutter_frames=64) as plan:
        d = torch.from_numpy(x).cuda()
        for bad in (d[:16].contiguous(), d):             # fewer than 32 frames; more than clutter_frames
            with pytest.raises(UlmRcaError):
                plan.clutter_filter(bad, 3)
        with pytest.raises(UlmRcaError):
            plan.clutter_filter(d[:64].contiguous(), 25)
    with pytest.raises(UlmRcaError):
        Plan(**rounded_kwargs(cfg), clutter_frames=321)
    with Plan(**rounded_kwargs(cfg)) as plan:
        with pytest.raises(ValueError):
            plan.clutter_filter(torch.from_numpy(x).cuda(), 3)


def test_config2_ensemble_size(torch_cuda):
    """The size bench.py times: 300 frames x 22 slices of 180 x 164 px (1.56 GB of slices).  Every event's covariance
    and eigenvalues against the oracle; the filtered slices of three events (first, a middle one, last) element by
    element."""
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan
    cfg = synth.config(2).with_(compound=0)
    kw = rounded_kwargs(cfg)
    p = oracle.OracleParams(**kw)
    n_pix = n_pix_list(cfg)
    x = synth.clutter_ensemble(300, n_pix, seed=22, tissue_rank=4)
    rank = 4
    with Plan(**kw, clutter_frames=300) as plan:
        d_x = torch.from_numpy(x).cuda()
        out, lam, cov = plan.clutter_filter(d_x, rank, want_eigenvalues=True, want_covariance=True)
        torch.cuda.synchronize()
        print("CLUTTER cfg2 kernel times (split, gram, assemble, eig, project) ms:", plan.clutter_timing())
        lam, cov = lam.cpu().numpy(), cov.cpu().numpy()
        blocks = clutter.event_blocks(p)
        scale = np.abs(x).max()
        for e, (off, n) in enumerate(blocks):
            xe = x[:, off:off + n].astype(np.complex128)
            c_ref = clutter.covariance(xe)
            lam_ref, _ = clutter.eig_desc(c_ref)
            e_cov = np.abs(cov[e] - c_ref).max() / np.abs(c_ref).max()
            e_lam = np.abs(lam[e][:rank + 2] - lam_ref[:rank + 2]).max() / lam_ref[0]
            assert e_cov <= 1e-4 and e_lam <= 1e-4, (e, e_cov, e_lam)
            if e in (0, 11, 21):
                ref, _, _ = clutter.clutter_filter_stack(xe, rank)
                got = out[:, off:off + n].cpu().numpy()
                e_out = np.abs(got - ref).max() / scale
                print("CLUTTER cfg2 event %d: cov %.2e eigenvalues %.2e filtered %.2e gap %.1f" % (e, e_cov, e_lam, e_out, lam_ref[rank - 1] / lam_ref[rank]))
                assert e_out <= 1e-4

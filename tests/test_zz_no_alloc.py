"""ulm_rca_localize_static -- the localization entry point that allocates nothing (its one scratch buffer, the per-frame
maximum, is a file-scope device array; include/ulm_rca.h) -- against the existing plan-based path ulm_rca_localize on the
same planes, on two calls in a row.  The second call uses much weaker planes, so a scratch array that kept the first
call's maxima would threshold every localization away.  Tolerances are those of tests/test_gpu_localize.py: count exact,
positions 1e-3 px, NCC 1e-4, intensity 1e-5 relative (the order inside a plane is not fixed: both lists are sorted).
This file is collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

import synth
from helpers import rounded_kwargs
from synth import centred_grid

pytestmark = pytest.mark.gpu
SIG = (1.8, 1.4)
NX, NY, NZ, BLOCK, CAP = 70, 40, 131, 8, 16
THR, NCC_MIN = 0.2, 0.7


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2511_21647_b200 import build
    build.build()
    return torch


def plan_kwargs():
    d = synth.LAMBDA_M / 2
    cfg = synth.config(0).with_(n_rows=24, n_cols=20, pitch=0.3e-3, n_samples=900, compound=0, n_frames=1,
                                row_tx_angles=(0.0,), col_tx_angles=(0.05,),
                                grid_xz=centred_grid(NX, d, NZ, 6e-3, d), grid_yz=centred_grid(NY, d, NZ, 6e-3, d))
    return rounded_kwargs(cfg)


def compare(loc_a, count_a, loc_b, count_b):
    assert np.array_equal(count_a, count_b)
    total = 0
    for f in range(count_a.shape[0]):
        for pl in range(count_a.shape[1]):
            n = min(int(count_a[f, pl]), CAP)
            a, b = sorted(loc_a[f, pl, :n].tolist()), sorted(loc_b[f, pl, :n].tolist())
            for g, o in zip(a, b):
                assert abs(g[0] - o[0]) <= 1e-3 and abs(g[1] - o[1]) <= 1e-3
                assert abs(g[2] - o[2]) <= 1e-4
                assert abs(g[3] - o[3]) <= 1e-5 * max(o[3], 1e-30)
            total += n
    return total


def test_static_scratch_matches_plan_path_twice(torch_cuda):
    torch = torch_cuda
    from paper_2511_21647_b200 import Plan, localize_static
    n_xz, n_yz = -(-NY // BLOCK), -(-NX // BLOCK)
    calls = []
    for seed, gain, n_frames in ((11, 1.0, 3), (12, 1e-3, 2)):
        planes = synth.bubble_planes(n_frames, n_xz, NX, n_yz, NY, NZ, seed, bubbles_per_plane=4, sigma=SIG)
        calls.append(torch.from_numpy((planes * gain).astype(np.complex64)).cuda())
    with Plan(**plan_kwargs(), stage2_block=BLOCK) as plan:
        assert (plan.n_planes_xz, plan.n_planes_yz) == (n_xz, n_yz)
        want = []
        for planes in calls:
            loc, count = plan.localize(planes, SIG[0], SIG[1], THR, NCC_MIN, CAP)
            torch.cuda.synchronize()
            want.append((loc.cpu().numpy(), count.cpu().numpy()))
    outs = [(torch.zeros((int(p.shape[0]), n_xz + n_yz, CAP, 4), dtype=torch.float32, device="cuda"),
             torch.full((int(p.shape[0]), n_xz + n_yz), -7, dtype=torch.int32, device="cuda")) for p in calls]
    torch.cuda.synchronize()
    free_before = None
    for i, (planes, (loc, count)) in enumerate(zip(calls, outs)):
        if i == 1:
            free_before = torch.cuda.mem_get_info()[0]       # the first call may load the module lazily; the second must not move it
        localize_static(planes, NZ, n_xz, NX, n_yz, NY, loc, count, SIG[0], SIG[1], THR, NCC_MIN)
        torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "the no-allocation entry point changed the free device memory"
    for (loc, count), (loc_w, count_w) in zip(outs, want):
        total = compare(loc.cpu().numpy(), count.cpu().numpy(), loc_w, count_w)
        assert total > 0


def test_static_scratch_limit_and_arguments(torch_cuda):
    torch = torch_cuda
    from paper_2511_21647_b200 import UlmRcaError, localize_static
    from paper_2511_21647_b200.binding import LOCALIZE_STATIC_MAX_FRAMES
    n = LOCALIZE_STATIC_MAX_FRAMES + 1
    planes = torch.zeros((n, 12 * 16), dtype=torch.complex64, device="cuda")          # one 12 x 16 plane per frame
    loc = torch.zeros((n, 1, 2, 4), dtype=torch.float32, device="cuda")
    count = torch.zeros((n, 1), dtype=torch.int32, device="cuda")
    with pytest.raises(UlmRcaError, match="exceeds the static scratch"):
        localize_static(planes, 16, 1, 12, 0, 0, loc, count, SIG[0], SIG[1], THR, NCC_MIN)
    # the limit itself is accepted; all-zero planes: nothing found
    localize_static(planes[:-1], 16, 1, 12, 0, 0, loc[:-1], count[:-1], SIG[0], SIG[1], THR, NCC_MIN)
    torch.cuda.synchronize()
    assert int(count.abs().sum()) == 0
    with pytest.raises(UlmRcaError, match="geometry"):          # no planes at all
        localize_static(torch.zeros((1, 0), dtype=torch.complex64, device="cuda"), 16, 0, 0, 0, 0,
                        torch.zeros((1, 0, 2, 4), dtype=torch.float32, device="cuda"),
                        torch.zeros((1, 0), dtype=torch.int32, device="cuda"), SIG[0], SIG[1], THR, NCC_MIN)

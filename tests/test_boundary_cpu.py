"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every symbol
include/ulm_rca.h declares, and refuses to run without a CUDA device (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2511_21647_b200 import build, binding
    build.build()
    return binding.load()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "ulm_rca.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ulm_rca_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    from paper_2511_21647_b200 import binding
    syms = declared_symbols()
    assert set(syms) == set(binding.EXPORTS), (syms, binding.EXPORTS)
    for s in syms:
        assert getattr(lib, s) is not None


def test_library_is_sm_100a_only():
    import subprocess
    from paper_2511_21647_b200 import binding
    out = subprocess.run(["cuobjdump", "--list-elf", binding.library_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in out and not re.search(r"sm_(?!100a)\d+", out), out


def test_null_and_invalid_arguments_are_status_codes(lib):
    from paper_2511_21647_b200 import binding as b
    assert lib.ulm_rca_plan_create(None, None, 0, None, 0, 1540.0, 20e6, 5e6, None, None, None, None) == b.EINVAL
    h = ctypes.c_void_p(123)
    st = lib.ulm_rca_plan_create(None, None, 0, None, 0, 1540.0, 20e6, 5e6, None, None, None, ctypes.byref(h))
    assert st == b.EINVAL and not h.value
    assert b"NULL" in lib.ulm_rca_last_error()
    assert lib.ulm_rca_beamform(None, None, 1, None, None) == b.EINVAL
    assert lib.ulm_rca_beamform_volume(None, None, 1, None, None) == b.EINVAL
    assert lib.ulm_rca_beamform_host(None, None, 1, None) == b.EINVAL
    assert lib.ulm_rca_plan_sizes(None, None, None, None) == b.EINVAL
    assert lib.ulm_rca_fp32_peak(None, None) == b.EINVAL
    lib.ulm_rca_plan_destroy(None)  # NULL-safe


def test_invalid_option_values(lib):
    import synth
    from paper_2511_21647_b200 import Plan, UlmRcaError
    from helpers import rounded_kwargs
    cfg = synth.config(0)
    bad = [dict(n_samples=1), dict(demod_taps=8), dict(compound=2), dict(input_kind=3), dict(fs=float("nan")),
           dict(channels_per_event=5), dict(grid_xz=(0, 0.0, 1e-4, 8, 1e-3, 1e-4, 0.0)),
           dict(grid_xz=(8, 0.0, 1e-4, 8, -1e-3, 1e-4, 0.0)), dict(row_tx_angles=[], col_tx_angles=[])]
    for kw in bad:
        with pytest.raises(UlmRcaError) as ei:
            Plan(**rounded_kwargs(cfg, **kw))
        assert ei.value.status == 1, kw


def test_no_cpu_fallback_without_a_device(lib):
    """On a box without a GPU a valid plan request must fail with ECUDA, not compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import synth
    from paper_2511_21647_b200 import Plan, UlmRcaError
    from helpers import rounded_kwargs
    with pytest.raises(UlmRcaError) as ei:
        Plan(**rounded_kwargs(synth.config(0)))
    assert ei.value.status == 3


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2511_21647_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower(), os.path.join(dirpath, f)

"""Writes tests/golden/tiny_projection.txt from the ORACLE ONLY (no CUDA code is imported).

The file freezes the oracle's output on a 4+4-element, 2+2-angle, RF-input case so that any later
change to oracle/ulm_oracle.c arithmetic is caught (and must be justified in its commit message).
The values are the oracle's own; what pins them to the mathematics is tests/test_oracle_pins.py.
Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import synth  # noqa: E402


def golden_case():
    d = synth.LAMBDA_M / 2
    cfg = synth.config(0).with_(
        n_rows=4, n_cols=4, n_samples=256, n_frames=1,
        row_tx_angles=tuple(np.radians([-3.0, 4.0])), col_tx_angles=tuple(np.radians([2.0, -5.0])),
        grid_xz=synth.centred_grid(3, d, 4, 5.0e-3, d, ref=0.2e-3),
        grid_yz=synth.centred_grid(2, 2 * d, 5, 5.2e-3, d / 2, ref=-0.1e-3),
        t_start=0.4e-6, f_number=1.1)
    n = np.arange(cfg.n_samples)
    ch = np.zeros(cfg.channel_shape, dtype=np.int16)
    for e in range(cfg.n_events):
        for c in range(cfg.channels_per_event):
            ch[0, e, c] = np.round(3000 * np.sin(0.37 * n + 0.9 * e + 0.31 * c) * np.cos(0.011 * n * (c + 1)))
    win = [1.0, 0.8, 0.6, 0.9, 0.5, 1.0, 0.7, 0.75]
    return cfg, ch, win


if __name__ == "__main__":
    cfg, ch, win = golden_case()
    kw = cfg.plan_kwargs()
    kw["elem_window"] = win
    out = oracle.beamform(oracle.OracleParams(**kw), ch)[0]
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_projection.txt")
    with open(path, "w") as f:
        f.write("# oracle output (re im per line), case = tests/golden/make_golden.py:golden_case()\n")
        f.write("# definition: SURVEY.md 8(c) steps 0-2 (PAPER.md:43-49 gives no formula)\n")
        for v in out:
            f.write("%.17e %.17e\n" % (v.real, v.imag))
    print("wrote", path, out.shape)

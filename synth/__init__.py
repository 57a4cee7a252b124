"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This package is the ONLY code both sides use.  It holds the workload configurations and a forward
echo simulator; it holds none of the beamformer's arithmetic and imports neither ``oracle`` nor
``paper_2511_21647_b200``.
"""
from .configs import RcaConfig, Scene, centred_grid, config, small_config, LAMBDA_M  # noqa: F401
from .scene import build, bubble_planes, clutter_ensemble, moving_speckle, random_channel, random_complex, render, scatterers  # noqa: F401

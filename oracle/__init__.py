"""fp64 CPU oracle of the RCA projection beamformer (Stage 1: ulm_oracle.c; Stage 2 + sum-projection: stage2.py)
-- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package (see oracle/ulm_oracle.h).  It imports nothing
from ``paper_2511_21647_b200`` and the CUDA path imports nothing from here.
"""
from .oracle import (  # noqa: F401
    OracleParams,
    beamform,
    build,
    das_points,
    demod_channel,
    fir_taps,
    threads,
    volume,
)
from . import stage2  # noqa: F401,E402
from . import clutter  # noqa: F401,E402
from . import motion  # noqa: F401,E402
from . import localize  # noqa: F401,E402

"""The five workload configurations of BASELINE.json (zero-based), as plain data.

Numbers come from BASELINE.json:configs and SURVEY.md 8(c) A9-A11 / 8(d); they follow the paper's
acquisition.  No beamforming arithmetic lives here.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Optional, Tuple

import numpy as np

C_MPS = 1540.0
FC_HZ = 5.0e6
LAMBDA_M = C_MPS / FC_HZ  # 0.308 mm


def centred_grid(n_lat: int, dlat: float, n_ax: int, z0: float, dz: float, ref: float = 0.0) -> tuple:
    """(n_lat, lat0, dlat, n_ax, z0, dz, ref) with the lateral axis centred on the array axis."""
    return (int(n_lat), -0.5 * (n_lat - 1) * dlat, float(dlat), int(n_ax), float(z0), float(dz), float(ref))


@dataclass(frozen=True)
class Scene:
    n_bubbles: int
    n_tissue: int
    tissue_gain_db: float
    half_width_m: float           # scatterers uniform in +-half_width in x and y
    z_range_m: Tuple[float, float]
    log_uniform_decades: float = 0.0   # bubble amplitudes log-uniform over this many decades
    moving: bool = False
    snr_db: float = 20.0


@dataclass(frozen=True)
class RcaConfig:
    name: str
    n_rows: int
    n_cols: int
    pitch: float
    fs: float
    n_samples: int
    row_tx_angles: Tuple[float, ...]
    col_tx_angles: Tuple[float, ...]
    grid_xz: tuple
    grid_yz: tuple
    n_frames: int
    scene: Scene
    seed: int
    fc: float = FC_HZ
    c: float = C_MPS
    frame_rate_hz: float = 400.0
    t_start: float = 0.0
    input_kind: int = 0
    all_channels: bool = True
    f_number: float = 0.0
    compound: int = 1
    volume: bool = False          # config 4: beamform the full 3-D volume instead of projections
    t0: Optional[Tuple[float, ...]] = None
    elem_window: Optional[Tuple[float, ...]] = None
    demod_taps: int = 0

    @property
    def n_events(self) -> int:
        return len(self.row_tx_angles) + len(self.col_tx_angles)

    @property
    def channels_per_event(self) -> int:
        return self.n_rows + self.n_cols if self.all_channels else max(self.n_rows, self.n_cols)

    @property
    def channel_shape(self) -> tuple:
        s = (self.n_frames, self.n_events, self.channels_per_event, self.n_samples)
        return s + (2,) if self.input_kind == 1 else s

    def plan_kwargs(self) -> dict:
        """Keyword arguments understood by both oracle.OracleParams and the CUDA binding's Plan."""
        return dict(n_rows=self.n_rows, n_cols=self.n_cols, pitch=self.pitch,
                    row_tx_angles=list(self.row_tx_angles), col_tx_angles=list(self.col_tx_angles),
                    c=self.c, fs=self.fs, fc=self.fc, grid_xz=self.grid_xz, grid_yz=self.grid_yz,
                    n_samples=self.n_samples, input_kind=self.input_kind,
                    channels_per_event=self.channels_per_event, t_start=self.t_start,
                    t0=None if self.t0 is None else list(self.t0), f_number=self.f_number,
                    elem_window=None if self.elem_window is None else list(self.elem_window),
                    demod_taps=self.demod_taps, compound=self.compound)

    def gather_samples_per_frame(self) -> int:
        """pixel x element x angle terms per frame."""
        if self.volume:
            nvox = self.grid_xz[0] * self.grid_yz[0] * self.grid_xz[3]
            return nvox * (len(self.row_tx_angles) * self.n_cols + len(self.col_tx_angles) * self.n_rows)
        return (self.grid_xz[0] * self.grid_xz[3] * len(self.row_tx_angles) * self.n_cols +
                self.grid_yz[0] * self.grid_yz[3] * len(self.col_tx_angles) * self.n_rows)

    def with_(self, **kw) -> "RcaConfig":
        return replace(self, **kw)


def _angles(n: int, max_deg: float) -> Tuple[float, ...]:
    return tuple(float(math.radians(a)) for a in np.linspace(-max_deg, max_deg, n))


def config(index: int) -> RcaConfig:
    """BASELINE.json:configs[index]."""
    if index == 0:
        d = LAMBDA_M / 2
        g = centred_grid(64, d, 96, 5e-3, d)
        return RcaConfig(name="cfg0-tiny", n_rows=32, n_cols=32, pitch=0.3e-3, fs=20e6, n_samples=1024,
                         row_tx_angles=_angles(3, 5.0), col_tx_angles=_angles(3, 5.0),
                         grid_xz=g, grid_yz=g, n_frames=2, seed=0,
                         scene=Scene(n_bubbles=10, n_tissue=0, tissue_gain_db=0.0, half_width_m=4.8e-3,
                                     z_range_m=(5e-3, 20e-3), log_uniform_decades=1.0))
    full_scene = Scene(n_bubbles=200, n_tissue=5000, tissue_gain_db=30.0, half_width_m=13.7e-3,
                       z_range_m=(20e-3, 45e-3))
    if index in (1, 2, 4):
        d = LAMBDA_M / 2
        g = centred_grid(180, d, 164, 20e-3, d)
        base = RcaConfig(name="cfg1-frame", n_rows=128, n_cols=128, pitch=0.214e-3, fs=20e6,
                         n_samples=2048, row_tx_angles=_angles(11, 10.0), col_tx_angles=_angles(11, 10.0),
                         grid_xz=g, grid_yz=g, n_frames=1, seed=1, scene=full_scene)
        if index == 1:
            return base
        if index == 2:
            return base.with_(name="cfg2-ensemble", n_frames=300, seed=2,
                              scene=replace(full_scene, moving=True))
        return base.with_(name="cfg4-volume", volume=True, seed=1)
    if index == 3:
        d = LAMBDA_M / 4
        g = centred_grid(360, d, 328, 20e-3, d)
        return RcaConfig(name="cfg3-fine", n_rows=128, n_cols=128, pitch=0.214e-3, fs=40e6, n_samples=4096,
                         row_tx_angles=_angles(11, 10.0), col_tx_angles=_angles(11, 10.0),
                         grid_xz=g, grid_yz=g, n_frames=300, seed=3,
                         scene=replace(full_scene, moving=True))
    raise ValueError("config index must be 0..4")


def small_config(**kw) -> RcaConfig:
    """A few-element variant of config 0 for closed-form and brute-force pins."""
    return config(0).with_(**kw)

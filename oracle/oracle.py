"""ctypes wrapper of oracle/ulm_oracle.c (TEST INFRASTRUCTURE; see ulm_oracle.h).

Argument marshalling only: every number the oracle produces is computed in ulm_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ulm_oracle.c")
_HDR = os.path.join(_HERE, "ulm_oracle.h")
_LIB = os.path.join(_HERE, "libulm_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile ulm_oracle.c with gcc (fp64, no fast-math, FP contraction off)."""
    stale = (not os.path.exists(_LIB)) or any(
        os.path.getmtime(s) > os.path.getmtime(_LIB) for s in (_SRC, _HDR)
    )
    if force or stale:
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
               "-Wall", "-Wextra", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


class _Grid(C.Structure):
    _fields_ = [("n_lat", C.c_int32), ("lat0", C.c_double), ("dlat", C.c_double),
                ("n_ax", C.c_int32), ("z0", C.c_double), ("dz", C.c_double), ("ref", C.c_double)]


class _Params(C.Structure):
    _fields_ = [("n_rows", C.c_int32), ("n_cols", C.c_int32), ("pitch", C.c_double),
                ("n_row_tx", C.c_int32), ("n_col_tx", C.c_int32),
                ("row_tx_angles", C.POINTER(C.c_double)), ("col_tx_angles", C.POINTER(C.c_double)),
                ("c", C.c_double), ("fs", C.c_double), ("fc", C.c_double),
                ("xz", _Grid), ("yz", _Grid),
                ("input_kind", C.c_int32), ("channels_per_event", C.c_int32),
                ("n_samples", C.c_int32), ("t_start", C.c_double),
                ("t0", C.POINTER(C.c_double)), ("f_number", C.c_double),
                ("elem_window", C.POINTER(C.c_double)), ("demod_taps", C.c_int32),
                ("compound", C.c_int32)]


def _load():
    global _lib
    if _lib is None:
        build()
        lib = C.CDLL(_LIB)
        lib.ulm_oracle_threads.restype = C.c_int
        lib.ulm_oracle_fir.restype = C.c_int
        lib.ulm_oracle_fir.argtypes = [C.POINTER(_Params), C.POINTER(C.c_double), C.c_int]
        lib.ulm_oracle_demod_channel.restype = C.c_int
        lib.ulm_oracle_demod_channel.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_void_p]
        lib.ulm_oracle_out_per_frame.restype = C.c_int64
        lib.ulm_oracle_out_per_frame.argtypes = [C.POINTER(_Params)]
        lib.ulm_oracle_beamform.restype = C.c_int
        lib.ulm_oracle_beamform.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_int32, C.c_void_p]
        lib.ulm_oracle_das_points.restype = C.c_int
        lib.ulm_oracle_das_points.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_void_p, C.c_int64,
                                              C.c_void_p, C.c_void_p]
        _lib = lib
    return _lib


@dataclass
class OracleParams:
    """Mirror of ulm_oracle_params.  Grids are (n_lat, lat0, dlat, n_ax, z0, dz, ref) tuples."""
    n_rows: int
    n_cols: int
    pitch: float
    row_tx_angles: Sequence[float]
    col_tx_angles: Sequence[float]
    c: float
    fs: float
    fc: float
    grid_xz: tuple
    grid_yz: tuple
    n_samples: int
    input_kind: int = 0
    channels_per_event: Optional[int] = None
    t_start: float = 0.0
    t0: Optional[Sequence[float]] = None
    f_number: float = 0.0
    elem_window: Optional[Sequence[float]] = None
    demod_taps: int = 0
    compound: int = 1
    _keep: list = field(default_factory=list, repr=False)

    def c_struct(self) -> _Params:
        self._keep.clear()

        def arr(v):
            if v is None:
                return None
            a = np.ascontiguousarray(np.asarray(v, dtype=np.float64))
            self._keep.append(a)
            return a.ctypes.data_as(C.POINTER(C.c_double))

        cpe = self.channels_per_event if self.channels_per_event is not None else self.n_rows + self.n_cols
        if self.t0 is not None:
            assert len(self.t0) == len(self.row_tx_angles) + len(self.col_tx_angles)
        if self.elem_window is not None:
            assert len(self.elem_window) == self.n_cols + self.n_rows
        return _Params(self.n_rows, self.n_cols, float(self.pitch),
                       len(self.row_tx_angles), len(self.col_tx_angles),
                       arr(self.row_tx_angles), arr(self.col_tx_angles),
                       float(self.c), float(self.fs), float(self.fc),
                       _Grid(*self.grid_xz), _Grid(*self.grid_yz),
                       int(self.input_kind), int(cpe), int(self.n_samples), float(self.t_start),
                       arr(self.t0), float(self.f_number), arr(self.elem_window),
                       int(self.demod_taps), int(self.compound))

    @property
    def n_events(self) -> int:
        return len(self.row_tx_angles) + len(self.col_tx_angles)

    @property
    def cpe(self) -> int:
        return self.channels_per_event if self.channels_per_event is not None else self.n_rows + self.n_cols

    def channel_shape(self, n_frames: int) -> tuple:
        s = (n_frames, self.n_events, self.cpe, self.n_samples)
        return s + (2,) if self.input_kind == 1 else s


def threads() -> int:
    return int(_load().ulm_oracle_threads())


def fir_taps(p: OracleParams) -> np.ndarray:
    h = np.zeros(1025, dtype=np.float64)
    ps = p.c_struct()
    L = _load().ulm_oracle_fir(C.byref(ps), h.ctypes.data_as(C.POINTER(C.c_double)), h.size)
    if L < 0:
        raise ValueError("ulm_oracle_fir failed: %d" % L)
    return h[: 2 * L + 1].copy()


def demod_channel(p: OracleParams, rec: np.ndarray) -> np.ndarray:
    rec = np.ascontiguousarray(rec, dtype=np.int16)
    assert rec.size == p.n_samples * (2 if p.input_kind == 1 else 1)
    out = np.zeros(p.n_samples, dtype=np.complex128)
    ps = p.c_struct()
    rc = _load().ulm_oracle_demod_channel(C.byref(ps), rec.ctypes.data, out.ctypes.data)
    if rc:
        raise ValueError("ulm_oracle_demod_channel failed: %d" % rc)
    return out


def beamform(p: OracleParams, channel: np.ndarray) -> np.ndarray:
    """channel: int16 [frame][event][channel][sample] (+[2] for IQ input).  Returns complex128
    [frame][out_per_frame] in the layout documented in ulm_oracle.h."""
    channel = np.ascontiguousarray(channel, dtype=np.int16)
    n_frames = channel.shape[0]
    assert channel.shape == p.channel_shape(n_frames), (channel.shape, p.channel_shape(n_frames))
    ps = p.c_struct()
    per = int(_load().ulm_oracle_out_per_frame(C.byref(ps)))
    out = np.zeros((n_frames, per), dtype=np.complex128)
    rc = _load().ulm_oracle_beamform(C.byref(ps), channel.ctypes.data, n_frames, out.ctypes.data)
    if rc:
        raise ValueError("ulm_oracle_beamform failed: %d" % rc)
    return out


def split_projections(p: OracleParams, out_frame: np.ndarray):
    """One frame of compound=1 output -> (P_xz [n_lat][n_ax], P_yz [n_lat][n_ax])."""
    nxz = p.grid_xz[0] * p.grid_xz[3]
    return (out_frame[:nxz].reshape(p.grid_xz[0], p.grid_xz[3]),
            out_frame[nxz:].reshape(p.grid_yz[0], p.grid_yz[3]))


def das_points(p: OracleParams, channel_frame: np.ndarray, xyz: np.ndarray):
    """3-D DAS at arbitrary points of ONE frame.  Returns (V_RC, V_CR) complex128 [n_pts]."""
    channel_frame = np.ascontiguousarray(channel_frame, dtype=np.int16)
    assert channel_frame.shape == p.channel_shape(1)[1:]
    xyz = np.ascontiguousarray(xyz, dtype=np.float64).reshape(-1, 3)
    n = xyz.shape[0]
    v_rc = np.zeros(n, dtype=np.complex128)
    v_cr = np.zeros(n, dtype=np.complex128)
    ps = p.c_struct()
    rc = _load().ulm_oracle_das_points(C.byref(ps), channel_frame.ctypes.data, xyz.ctypes.data, n,
                                       v_rc.ctypes.data, v_cr.ctypes.data)
    if rc:
        raise ValueError("ulm_oracle_das_points failed: %d" % rc)
    return v_rc, v_cr


def volume(p: OracleParams, channel_frame: np.ndarray, xs, ys, zs):
    """3-D DAS volume [x][y][z] of ONE frame on the given coordinate lists: (V_RC, V_CR)."""
    xs, ys, zs = (np.asarray(a, dtype=np.float64) for a in (xs, ys, zs))
    X, Y, Z = np.meshgrid(xs, ys, zs, indexing="ij")
    pts = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)
    v_rc, v_cr = das_points(p, channel_frame, pts)
    shp = (xs.size, ys.size, zs.size)
    return v_rc.reshape(shp), v_cr.reshape(shp)

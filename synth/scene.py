"""Seeded scatterer scenes and channel-data rendering (INPUT GENERATOR ONLY; recipe in DESIGN.md).

Scene kinematics: bubbles move on straight lines or circular arcs at 1-50 mm/s and
are born/die with Poisson(20) per frame; tissue scatterers share a 0.5 mm, 0.3 Hz axial oscillation.
Rendering of the echoes is done by synth/ulm_synth.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, Iterable, List, Optional

import numpy as np

from .configs import RcaConfig

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ulm_synth.c")
_LIB = os.path.join(_HERE, "libulm_synth.so")
_lib = None


class _Params(C.Structure):
    _fields_ = [("n_rows", C.c_int32), ("n_cols", C.c_int32), ("pitch", C.c_double),
                ("n_row_tx", C.c_int32), ("n_col_tx", C.c_int32),
                ("row_tx_angles", C.POINTER(C.c_double)), ("col_tx_angles", C.POINTER(C.c_double)),
                ("c", C.c_double), ("fs", C.c_double), ("fc", C.c_double),
                ("n_samples", C.c_int32), ("t_start", C.c_double), ("t0", C.POINTER(C.c_double)),
                ("all_channels", C.c_int32)]


def build(force: bool = False) -> str:
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_SRC) > os.path.getmtime(_LIB)
    if force or stale:
        subprocess.run(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", _LIB,
                        _SRC, "-lm"], check=True, cwd=_HERE)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = C.CDLL(_LIB)
        lib.ulm_synth_stats.restype = C.c_int
        lib.ulm_synth_stats.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_int64,
                                        C.POINTER(C.c_double), C.POINTER(C.c_double)]
        lib.ulm_synth_render.restype = C.c_int
        lib.ulm_synth_render.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_int64, C.c_double,
                                         C.c_double, C.c_uint64, C.c_int64, C.c_void_p]
        _lib = lib
    return _lib


def _params(cfg: RcaConfig, keep: list) -> _Params:
    def arr(v):
        if v is None:
            return None
        a = np.ascontiguousarray(np.asarray(v, dtype=np.float64))
        keep.append(a)
        return a.ctypes.data_as(C.POINTER(C.c_double))

    return _Params(cfg.n_rows, cfg.n_cols, cfg.pitch, len(cfg.row_tx_angles), len(cfg.col_tx_angles),
                   arr(cfg.row_tx_angles), arr(cfg.col_tx_angles), cfg.c, cfg.fs, cfg.fc,
                   cfg.n_samples, cfg.t_start, arr(cfg.t0), 1 if cfg.all_channels else 0)


def _rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[int(seed), int(stream)]))


def _uniform_points(rng, n, sc) -> np.ndarray:
    p = np.empty((n, 3))
    p[:, 0] = rng.uniform(-sc.half_width_m, sc.half_width_m, n)
    p[:, 1] = rng.uniform(-sc.half_width_m, sc.half_width_m, n)
    p[:, 2] = rng.uniform(sc.z_range_m[0], sc.z_range_m[1], n)
    return p


def _new_bubbles(rng, n, sc) -> Dict[str, np.ndarray]:
    """Birth state of n bubbles: position, unit direction, speed, arc flag, arc radius, arc normal."""
    pos = _uniform_points(rng, n, sc)
    d = rng.normal(size=(n, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True) + 1e-300
    q = rng.normal(size=(n, 3))
    q -= (q * d).sum(1, keepdims=True) * d          # unit vector orthogonal to the direction
    q /= np.linalg.norm(q, axis=1, keepdims=True) + 1e-300
    amp = 10.0 ** rng.uniform(-sc.log_uniform_decades, 0.0, n) if sc.log_uniform_decades > 0 else np.ones(n)
    return dict(pos0=pos, dir=d, side=q, speed=rng.uniform(1e-3, 50e-3, n),
                arc=rng.uniform(size=n) < 0.5, radius=rng.uniform(1e-3, 5e-3, n), amp=amp,
                age=np.zeros(n))


def _bubble_positions(b, dt) -> np.ndarray:
    """Position after age*dt seconds: straight line, or a circular arc of the given radius."""
    t = (b["age"] * dt)[:, None]
    straight = b["pos0"] + b["dir"] * b["speed"][:, None] * t
    ang = b["speed"][:, None] * t / b["radius"][:, None]
    arc = b["pos0"] + b["radius"][:, None] * (np.sin(ang) * b["dir"] + (1.0 - np.cos(ang)) * b["side"])
    return np.where(b["arc"][:, None], arc, straight)


def scatterers(cfg: RcaConfig, frames: Iterable[int]) -> Dict[int, np.ndarray]:
    """{frame: float64 [S][4] = (x, y, z, amplitude)} for the requested frames, simulated
    sequentially from frame 0 (seed = cfg.seed)."""
    sc = cfg.scene
    frames = sorted(set(int(f) for f in frames))
    rng = _rng(cfg.seed, 1)
    tissue = _uniform_points(rng, sc.n_tissue, sc)
    tissue_amp = np.full(sc.n_tissue, 10.0 ** (sc.tissue_gain_db / 20.0))
    bub = _new_bubbles(rng, sc.n_bubbles, sc)
    dt = 1.0 / cfg.frame_rate_hz
    out: Dict[int, np.ndarray] = {}
    last = frames[-1] if frames else -1
    for f in range(last + 1):
        if f in frames:
            tz = tissue.copy()
            if sc.moving:
                tz[:, 2] += 0.5e-3 * np.sin(2.0 * np.pi * 0.3 * f * dt)
            bp = _bubble_positions(bub, dt) if sc.moving else bub["pos0"]
            out[f] = np.concatenate([np.column_stack([bp, bub["amp"]]),
                                     np.column_stack([tz, tissue_amp])], axis=0)
        if sc.moving:
            bub["age"] = bub["age"] + 1.0
            n_die = min(int(rng.poisson(20)), bub["age"].size)
            keep = np.ones(bub["age"].size, dtype=bool)
            keep[rng.choice(bub["age"].size, size=n_die, replace=False)] = False
            born = _new_bubbles(rng, int(rng.poisson(20)), sc)
            bub = {k: np.concatenate([v[keep], born[k]], axis=0) for k, v in bub.items()}
    return out


def render(cfg: RcaConfig, frames: Optional[Iterable[int]] = None, noise: bool = True,
           scat: Optional[Dict[int, np.ndarray]] = None) -> np.ndarray:
    """int16 channel data [len(frames)][event][channel][sample] (RF) for the given frame indices
    (default: all cfg.n_frames).  Quantisation scale and noise level are fixed from frame 0:
    scale maps 1.25 x the noise-free max |value| of frame 0 to 8191; noise variance is the noise-free
    mean square of frame 0 / 10^(snr_db/10)."""
    assert cfg.input_kind == 0, "the echo model renders RF; IQ-input tests build their own data"
    frames = list(range(cfg.n_frames)) if frames is None else [int(f) for f in frames]
    sc = scat if scat is not None else scatterers(cfg, set(frames) | {0})   # scat: explicit {frame: [S][4]}
    lib = _load()
    keep: list = []
    ps = _params(cfg, keep)
    s0 = np.ascontiguousarray(sc[0] if 0 in sc else sc[frames[0]])
    mx, msq = C.c_double(), C.c_double()
    lib.ulm_synth_stats(C.byref(ps), s0.ctypes.data, s0.shape[0], C.byref(mx), C.byref(msq))
    scale = 8191.0 / (1.25 * mx.value) if mx.value > 0 else 1.0
    sigma = float(np.sqrt(msq.value / 10.0 ** (cfg.scene.snr_db / 10.0))) if noise else 0.0
    out = np.zeros((len(frames), cfg.n_events, cfg.channels_per_event, cfg.n_samples), dtype=np.int16)
    for i, f in enumerate(frames):
        s = np.ascontiguousarray(sc[f])
        lib.ulm_synth_render(C.byref(ps), s.ctypes.data, s.shape[0], scale, sigma, cfg.seed, f,
                             out[i].ctypes.data)
    return out


def random_channel(cfg: RcaConfig, n_frames: int, seed: int, amplitude: int = 2000) -> np.ndarray:
    """Band-unlimited random int16 data of the config's shape (for linearity / symmetry checks)."""
    rng = _rng(seed, 7)
    shape = (n_frames, cfg.n_events, cfg.channels_per_event, cfg.n_samples)
    if cfg.input_kind == 1:
        shape = shape + (2,)
    return rng.integers(-amplitude, amplitude + 1, size=shape, dtype=np.int16)


def random_complex(shape, seed: int, amplitude: float = 1.0) -> np.ndarray:
    """Seeded complex64 array (normal real and imaginary parts): stand-in for beamformed slices / images where a test
    of a later pipeline stage needs an input that does not come from either beamformer."""
    rng = _rng(seed, 11)
    return (amplitude * (rng.standard_normal(shape) + 1j * rng.standard_normal(shape))).astype(np.complex64)


def clutter_ensemble(n_t: int, n_pix_per_event, seed: int, tissue_rank: int = 3, tissue_gain_db: float = 30.0,
                     bubble_density: float = 0.01, noise: float = 0.05) -> np.ndarray:
    """Seeded complex64 slice stacks [n_t][sum of n_pix_per_event] shaped like clutter-dominated Stage-1 output (stand-in
    for the in-vivo slices of PAPER.md:53-59, which are not available): per event, `tissue_rank` strong components
    (smooth slow-time profile x fixed spatial speckle, tissue_gain_db above the bubbles, decaying 6 dB per component),
    sparse unit-amplitude "bubble" samples that change from frame to frame, and white noise."""
    rng = _rng(seed, 13)
    f = np.arange(n_t)[:, None]
    blocks = []
    for n in n_pix_per_event:
        x = noise * (rng.standard_normal((n_t, n)) + 1j * rng.standard_normal((n_t, n)))
        hit = rng.random((n_t, n)) < bubble_density
        x = x + hit * np.exp(2j * np.pi * rng.random((n_t, n)))
        for m in range(tissue_rank):
            gain = 10.0 ** ((tissue_gain_db - 6.0 * m) / 20.0)
            drift = np.exp(2j * np.pi * (0.3 * (m + 1) * np.sin(2 * np.pi * (m + 1) * f / (2.5 * n_t) + rng.random()) + rng.random()))
            speckle = (rng.standard_normal(n) + 1j * rng.standard_normal(n)) / np.sqrt(2.0)
            x = x + gain * drift * speckle[None, :]
        blocks.append(x)
    return np.concatenate(blocks, axis=1).astype(np.complex64)


def moving_speckle(n_frames: int, shapes, shifts, seed: int, correlation_px: float = 3.0, noise: float = 0.02) -> np.ndarray:
    """Seeded complex64 slices [n_frames][sum of n_lat * n_ax over `shapes`] whose B-mode images are one smooth random
    speckle field per event, displaced in frame f by shifts[f] = (lateral px, axial px) (sub-pixel displacement by the
    Fourier shift theorem on a larger canvas, then cropped) plus a little independent noise: stand-in for the slices of a
    slowly moving organ."""
    rng = _rng(seed, 17)
    out = []
    for (nl, nz) in shapes:
        m1, m2 = 2 * nl + 32, 2 * nz + 32
        k1, k2 = np.fft.fftfreq(m1)[:, None], np.fft.fftfreq(m2)[None, :]
        spec = np.fft.fft2(rng.standard_normal((m1, m2)) + 1j * rng.standard_normal((m1, m2)))
        spec *= np.exp(-2.0 * (np.pi * correlation_px) ** 2 * (k1 ** 2 + k2 ** 2))          # Gaussian low-pass
        frames = []
        for f in range(n_frames):
            s1, s2 = shifts[f]
            img = np.fft.ifft2(spec * np.exp(-2j * np.pi * (k1 * s1 + k2 * s2)))
            crop = img[nl // 2 + 8:nl // 2 + 8 + nl, nz // 2 + 8:nz // 2 + 8 + nz]
            crop = crop / np.abs(crop).max() + noise * (rng.standard_normal((nl, nz)) + 1j * rng.standard_normal((nl, nz)))
            frames.append(crop.reshape(-1))
        out.append(np.stack(frames))
    return np.concatenate(out, axis=1).astype(np.complex64)


def bubble_planes(n_frames: int, n_planes_xz: int, nx: int, n_planes_yz: int, ny: int, nz: int, seed: int, bubbles_per_plane: int = 4,
                  sigma=(1.8, 1.4), noise: float = 0.01) -> np.ndarray:
    """Seeded complex64 projected planes [n_frames][layout of ulm_rca_stage2_project]: every plane holds a few Gaussian
    blobs (width `sigma` pixels along lateral / depth, amplitudes 0.3 .. 1, random phase) at random sub-pixel positions at
    least 9 pixels apart, plus weak complex noise: stand-in for separated microbubble planes."""
    rng = _rng(seed, 19)
    out = np.zeros((n_frames, (n_planes_xz * nx + n_planes_yz * ny) * nz), dtype=np.complex64)
    for f in range(n_frames):
        off = 0
        for (n_pl, nl) in ((n_planes_xz, nx), (n_planes_yz, ny)):
            for _ in range(n_pl):
                img = noise * (rng.standard_normal((nl, nz)) + 1j * rng.standard_normal((nl, nz)))
                ll, zz = np.meshgrid(np.arange(nl), np.arange(nz), indexing="ij")
                placed = []
                for _b in range(bubbles_per_plane):
                    for _try in range(50):
                        c = (rng.uniform(7, nl - 8), rng.uniform(7, nz - 8))
                        if all((c[0] - q[0]) ** 2 + (c[1] - q[1]) ** 2 >= 81 for q in placed):
                            placed.append(c)
                            break
                    else:
                        continue
                    amp = rng.uniform(0.3, 1.0) * np.exp(2j * np.pi * rng.random())
                    img = img + amp * np.exp(-((ll - c[0]) ** 2) / (2 * sigma[0] ** 2) - ((zz - c[1]) ** 2) / (2 * sigma[1] ** 2))
                out[f, off:off + nl * nz] = img.reshape(-1)
                off += nl * nz
    return out

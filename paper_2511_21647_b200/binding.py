"""Thin ctypes binding of include/ulm_rca.h -- argument marshalling only.

Every step of the hot path runs inside libulm_rca.so (hand-written CUDA for sm_100a).  PyTorch is used
for device memory and streams only.  There is no fallback: if the library is missing or there is no
CUDA device, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libulm_rca.so")
_lib = None

OK, EINVAL, ENOMEM, ECUDA, EUNSUPPORTED = range(5)
_STATUS = {1: "EINVAL", 2: "ENOMEM", 3: "ECUDA", 4: "EUNSUPPORTED"}

EXPORTS = ["ulm_rca_plan_create", "ulm_rca_beamform", "ulm_rca_beamform_volume", "ulm_rca_beamform_host",
           "ulm_rca_plan_sizes", "ulm_rca_plan_info", "ulm_rca_plan_timing", "ulm_rca_fp32_peak", "ulm_rca_ring_probe", "ulm_rca_fold_probe",
           "ulm_rca_stage2_project", "ulm_rca_stage2_sizes", "ulm_rca_stage2_timing",
           "ulm_rca_clutter_filter", "ulm_rca_clutter_timing", "ulm_rca_motion_estimate", "ulm_rca_motion_timing", "ulm_rca_localize", "ulm_rca_localize_static",
           "ulm_rca_plan_destroy",
           "ulm_rca_last_error"]


class UlmRcaError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__("ulm_rca: %s: %s" % (_STATUS.get(status, status), text))
        self.status = status


class Geometry(C.Structure):
    _fields_ = [("n_rows", C.c_int32), ("n_cols", C.c_int32), ("pitch_m", C.c_float)]


class Grid(C.Structure):
    _fields_ = [("n_lat", C.c_int32), ("lat0_m", C.c_float), ("dlat_m", C.c_float),
                ("n_ax", C.c_int32), ("z0_m", C.c_float), ("dz_m", C.c_float), ("ref_m", C.c_float)]


class LocalizeParams(C.Structure):
    _fields_ = [("sigma_lat_px", C.c_float), ("sigma_ax_px", C.c_float), ("threshold_rel", C.c_float), ("ncc_min", C.c_float),
                ("capacity", C.c_int32)]


class Options(C.Structure):
    _fields_ = [("input_kind", C.c_int32), ("channels_per_event", C.c_int32), ("n_samples", C.c_int32),
                ("t_start_s", C.c_float), ("t0_s", C.POINTER(C.c_float)), ("f_number", C.c_float),
                ("elem_window", C.POINTER(C.c_float)), ("demod_taps", C.c_int32), ("compound", C.c_int32),
                ("max_frames", C.c_int32), ("build_volume", C.c_int32), ("kernel", C.c_int32),
                ("precision", C.c_int32), ("no_timing", C.c_int32), ("stage2_block", C.c_int32), ("clutter_frames", C.c_int32), ("motion_frames", C.c_int32)]


def library_path() -> str:
    return _LIB_PATH


def load() -> C.CDLL:
    """dlopen libulm_rca.so (built by paper_2511_21647_b200.build) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise RuntimeError("libulm_rca.so is not built: run `python -m paper_2511_21647_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(_LIB_PATH)
    vp, i32 = C.c_void_p, C.c_int32
    lib.ulm_rca_plan_create.restype = C.c_int
    lib.ulm_rca_plan_create.argtypes = [C.POINTER(Geometry), C.POINTER(C.c_float), i32, C.POINTER(C.c_float), i32,
                                        C.c_float, C.c_float, C.c_float, C.POINTER(Grid), C.POINTER(Grid),
                                        C.POINTER(Options), C.POINTER(vp)]
    lib.ulm_rca_beamform.restype = C.c_int
    lib.ulm_rca_beamform.argtypes = [vp, vp, i32, vp, vp]
    lib.ulm_rca_beamform_volume.restype = C.c_int
    lib.ulm_rca_beamform_volume.argtypes = [vp, vp, i32, vp, vp]
    lib.ulm_rca_beamform_host.restype = C.c_int
    lib.ulm_rca_beamform_host.argtypes = [vp, vp, i32, vp]
    lib.ulm_rca_plan_sizes.restype = C.c_int
    lib.ulm_rca_plan_sizes.argtypes = [vp, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
    lib.ulm_rca_plan_info.restype = C.c_int
    lib.ulm_rca_plan_info.argtypes = [vp, C.POINTER(C.c_int64), i32]
    lib.ulm_rca_plan_timing.restype = C.c_int
    lib.ulm_rca_plan_timing.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.ulm_rca_stage2_project.restype = C.c_int
    lib.ulm_rca_stage2_project.argtypes = [vp, vp, i32, vp, vp]
    lib.ulm_rca_stage2_sizes.restype = C.c_int
    lib.ulm_rca_stage2_sizes.argtypes = [vp, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t), C.POINTER(i32), C.POINTER(i32)]
    lib.ulm_rca_stage2_timing.restype = C.c_int
    lib.ulm_rca_stage2_timing.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.ulm_rca_clutter_filter.restype = C.c_int
    lib.ulm_rca_clutter_filter.argtypes = [vp, vp, i32, i32, vp, vp, vp, vp]
    lib.ulm_rca_clutter_timing.restype = C.c_int
    lib.ulm_rca_clutter_timing.argtypes = [vp, C.POINTER(C.c_double)]
    lib.ulm_rca_motion_estimate.restype = C.c_int
    lib.ulm_rca_motion_estimate.argtypes = [vp, vp, i32, i32, vp, vp, vp]
    lib.ulm_rca_motion_timing.restype = C.c_int
    lib.ulm_rca_motion_timing.argtypes = [vp, C.POINTER(C.c_double)]
    lib.ulm_rca_localize.restype = C.c_int
    lib.ulm_rca_localize.argtypes = [vp, vp, i32, C.POINTER(LocalizeParams), vp, vp, vp]
    lib.ulm_rca_localize_static.restype = C.c_int
    lib.ulm_rca_localize_static.argtypes = [vp, i32, i32, i32, i32, i32, i32, C.POINTER(LocalizeParams), vp, vp, vp]
    lib.ulm_rca_fp32_peak.restype = C.c_int
    lib.ulm_rca_fp32_peak.argtypes = [C.POINTER(C.c_double), vp]
    lib.ulm_rca_ring_probe.restype = C.c_int
    lib.ulm_rca_ring_probe.argtypes = [i32, C.c_float, C.POINTER(C.c_float), C.POINTER(C.c_float), i32, C.c_float,
                                       C.c_float, C.c_float, C.POINTER(Grid), C.POINTER(i32), C.POINTER(i32),
                                       C.POINTER(i32), C.POINTER(i32)]
    lib.ulm_rca_fold_probe.restype = C.c_int
    lib.ulm_rca_fold_probe.argtypes = [C.POINTER(C.c_float), C.POINTER(C.c_float), i32, C.c_float, C.c_float,
                                       C.POINTER(Grid), C.POINTER(i32)]
    lib.ulm_rca_plan_destroy.restype = None
    lib.ulm_rca_plan_destroy.argtypes = [vp]
    lib.ulm_rca_last_error.restype = C.c_char_p
    lib.ulm_rca_last_error.argtypes = []
    _lib = lib
    return lib


def _check(status: int):
    if status != OK:
        raise UlmRcaError(status, load().ulm_rca_last_error().decode("utf-8", "replace"))


def _farr(v):
    if v is None:
        return None, None
    a = np.ascontiguousarray(np.asarray(v, dtype=np.float32))
    return a, a.ctypes.data_as(C.POINTER(C.c_float))


INFO_KEYS = ["n_lo", "l_row", "iq_scratch_bytes", "kernel", "frames_per_thread", "tile_pixels", "window",
             "stages", "tiles_xz", "smem_bytes", "launches_last_call", "tiles_yz", "precision", "scratch_bytes_per_sample", "host_upload_bytes_per_frame", "events_executed",
             "stage2_taps", "stage2_tile_cols", "window_two_groups", "stages_two_groups", "tiles_xz_two_groups", "tiles_yz_two_groups", "volume_mirror_pairs"]


LOCALIZE_STATIC_MAX_FRAMES = 4096        # ULM_RCA_LOCALIZE_STATIC_MAX_FRAMES of include/ulm_rca.h


def localize_static(planes, n_z: int, n_planes_xz: int, n_lat_xz: int, n_planes_yz: int, n_lat_yz: int, loc, count,
                    sigma_lat_px: float, sigma_ax_px: float, threshold_rel: float, ncc_min: float, stream=None):
    """ulm_rca_localize_static: the localization without a plan and without any allocation.  planes: contiguous complex64
    CUDA tensor [frame][planes of a frame]; loc (float32 [frame][plane][capacity][4]) and count (int32 [frame][plane]) are
    the CALLER's CUDA tensors (nothing is allocated here either); all calls on a device share one static scratch array,
    so calls that may overlap on the GPU race (see include/ulm_rca.h)."""
    import torch
    n_pl = int(n_planes_xz) + int(n_planes_yz)
    per_frame = (int(n_planes_xz) * int(n_lat_xz) + int(n_planes_yz) * int(n_lat_yz)) * int(n_z)
    if not (planes.is_cuda and planes.dtype == torch.complex64 and planes.is_contiguous() and planes.dim() == 2
            and planes.shape[1] == per_frame):
        raise ValueError("planes must be a contiguous complex64 CUDA tensor [frame][%d]" % per_frame)
    n = int(planes.shape[0])
    if not (loc.is_cuda and loc.dtype == torch.float32 and loc.is_contiguous() and loc.dim() == 4 and loc.shape[0] == n
            and loc.shape[1] == n_pl and loc.shape[3] == 4 and loc.device == planes.device):
        raise ValueError("loc must be a contiguous float32 CUDA tensor [frame][plane][capacity][4] on the planes' device")
    if not (count.is_cuda and count.dtype == torch.int32 and count.is_contiguous() and tuple(count.shape) == (n, n_pl)
            and count.device == planes.device):
        raise ValueError("count must be a contiguous int32 CUDA tensor [frame][plane] on the planes' device")
    prm = LocalizeParams(float(sigma_lat_px), float(sigma_ax_px), float(threshold_rel), float(ncc_min), int(loc.shape[2]))
    s = stream if stream is not None else torch.cuda.current_stream(planes.device)
    with torch.cuda.device(planes.device):
        _check(load().ulm_rca_localize_static(C.c_void_p(planes.data_ptr()), n, int(n_z), int(n_planes_xz), int(n_lat_xz),
                                              int(n_planes_yz), int(n_lat_yz), C.byref(prm), C.c_void_p(loc.data_ptr()),
                                              C.c_void_p(count.data_ptr()), C.c_void_p(s.cuda_stream)))
    return loc, count


class Plan:
    """ulm_rca_plan_create / ulm_rca_beamform / ulm_rca_plan_destroy with torch tensors as device memory.

    Grids are (n_lat, lat0_m, dlat_m, n_ax, z0_m, dz_m, ref_m) tuples; angles in radians.
    """

    def __init__(self, n_rows: int, n_cols: int, pitch: float, row_tx_angles: Sequence[float],
                 col_tx_angles: Sequence[float], c: float, fs: float, fc: float, grid_xz: tuple, grid_yz: tuple,
                 n_samples: int, input_kind: int = 0, channels_per_event: Optional[int] = None,
                 t_start: float = 0.0, t0: Optional[Sequence[float]] = None, f_number: float = 0.0,
                 elem_window: Optional[Sequence[float]] = None, demod_taps: int = 0, compound: int = 1,
                 max_frames: int = 0, build_volume: bool = False, kernel: int = 0, precision: int = 0,
                 no_timing: bool = False, stage2_block: int = 0, clutter_frames: int = 0,
                 motion_frames: int = 0):
        lib = load()
        self._h = C.c_void_p()
        geo = Geometry(n_rows, n_cols, pitch)
        ra, rp = _farr(list(row_tx_angles))
        ca, cp = _farr(list(col_tx_angles))
        ta, tp = _farr(t0)
        wa, wp = _farr(elem_window)
        if t0 is not None and len(t0) != len(row_tx_angles) + len(col_tx_angles):
            raise ValueError("t0 must have one entry per event")
        if elem_window is not None and len(elem_window) != n_rows + n_cols:
            raise ValueError("elem_window must have n_cols + n_rows entries")
        opt = Options(int(input_kind), int(channels_per_event or 0), int(n_samples), float(t_start), tp,
                      float(f_number), wp, int(demod_taps), int(compound), int(max_frames),
                      1 if build_volume else 0, int(kernel), int(precision), 1 if no_timing else 0, int(stage2_block), int(clutter_frames), int(motion_frames))
        gx, gy = Grid(*grid_xz), Grid(*grid_yz)
        _check(lib.ulm_rca_plan_create(C.byref(geo), rp, len(row_tx_angles), cp, len(col_tx_angles),
                                       float(c), float(fs), float(fc), C.byref(gx), C.byref(gy), C.byref(opt),
                                       C.byref(self._h)))
        a, b, v = C.c_size_t(), C.c_size_t(), C.c_size_t()
        _check(lib.ulm_rca_plan_sizes(self._h, C.byref(a), C.byref(b), C.byref(v)))
        self.channel_bytes_per_frame, self.out_bytes_per_frame, self.volume_bytes_per_frame = a.value, b.value, v.value
        self.input_kind, self.compound = int(input_kind), int(compound)
        self.volume_shape = (grid_xz[0], grid_yz[0], grid_xz[3])
        self.grid_xz, self.grid_yz = tuple(grid_xz), tuple(grid_yz)
        self.n_row_tx, self.n_col_tx = len(row_tx_angles), len(col_tx_angles)
        import torch
        self.device_index = torch.cuda.current_device()      # the plan belongs to the device current at creation
        self.clutter_frames = int(clutter_frames)
        self.motion_frames = int(motion_frames)
        self.n_events = len(row_tx_angles) + len(col_tx_angles)
        self.slices_complex_per_frame = (len(row_tx_angles) * grid_xz[0] * grid_xz[3] + len(col_tx_angles) * grid_yz[0] * grid_yz[3])
        self.stage2_block = int(stage2_block)
        if self.stage2_block:
            sb, pb, nxz, nyz = C.c_size_t(), C.c_size_t(), C.c_int32(), C.c_int32()
            _check(lib.ulm_rca_stage2_sizes(self._h, C.byref(sb), C.byref(pb), C.byref(nxz), C.byref(nyz)))
            self.slices_bytes_per_frame, self.planes_bytes_per_frame = sb.value, pb.value
            self.n_planes_xz, self.n_planes_yz = nxz.value, nyz.value

    # -- lifetime -------------------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load().ulm_rca_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- facts ----------------------------------------------------------------------------------------
    def info(self) -> dict:
        v = (C.c_int64 * len(INFO_KEYS))()
        _check(load().ulm_rca_plan_info(self._h, v, len(INFO_KEYS)))
        return dict(zip(INFO_KEYS, [int(x) for x in v]))

    def timing(self, n_calls: int = 1) -> tuple:
        """(demod_ms, das_ms): mean device time per call of the kernels of the last n_calls beamform() calls."""
        d, g = C.c_double(), C.c_double()
        _check(load().ulm_rca_plan_timing(self._h, int(n_calls), C.byref(d), C.byref(g)))
        return d.value, g.value

    @property
    def out_complex_per_frame(self) -> int:
        return self.out_bytes_per_frame // 8

    # -- calls ----------------------------------------------------------------------------------------
    def _stream_ptr(self, stream):
        import torch
        s = stream if stream is not None else torch.cuda.current_stream()
        return C.c_void_p(s.cuda_stream)

    def _check_channel(self, channel) -> int:
        import torch
        if not (channel.is_cuda and channel.dtype == torch.int16 and channel.is_contiguous()):
            raise ValueError("channel must be a contiguous int16 CUDA tensor")
        if channel.device.index != self.device_index:
            raise ValueError("channel lives on cuda:%d, the plan on cuda:%d" % (channel.device.index, self.device_index))
        n_frames = int(channel.shape[0])
        if n_frames and channel.numel() * 2 != n_frames * self.channel_bytes_per_frame:
            raise ValueError("channel has %d bytes per frame, plan expects %d" %
                             (channel.numel() * 2 // n_frames, self.channel_bytes_per_frame))
        return n_frames

    def _check_out(self, out, numel: int):
        import torch
        if not (out.is_cuda and out.dtype == torch.complex64 and out.is_contiguous() and out.numel() == numel
                and out.device.index == self.device_index):
            raise ValueError("out must be a contiguous complex64 CUDA tensor of the plan's size on the plan's device")

    def beamform(self, channel, out=None, stream=None):
        """channel: torch int16 CUDA tensor [frame][event][channel][sample] (+[2] for IQ input).
        Returns a torch complex64 CUDA tensor [frame][out_complex_per_frame]; asynchronous on `stream`."""
        import torch
        n_frames = self._check_channel(channel)
        if out is None:
            out = torch.empty((n_frames, self.out_complex_per_frame), dtype=torch.complex64, device=channel.device)
        else:
            self._check_out(out, n_frames * self.out_complex_per_frame)
        _check(load().ulm_rca_beamform(self._h, C.c_void_p(channel.data_ptr()), n_frames,
                                       C.c_void_p(out.data_ptr()), self._stream_ptr(stream)))
        return out

    def beamform_volume(self, channel, out=None, stream=None):
        """Full 3-D DAS comparator: returns complex64 [frame][x][y][z]."""
        import torch
        n_frames = self._check_channel(channel)
        if out is None:
            out = torch.empty((n_frames,) + self.volume_shape, dtype=torch.complex64, device=channel.device)
        else:
            self._check_out(out, n_frames * self.volume_bytes_per_frame // 8)
        _check(load().ulm_rca_beamform_volume(self._h, C.c_void_p(channel.data_ptr()), n_frames,
                                              C.c_void_p(out.data_ptr()), self._stream_ptr(stream)))
        return out

    def stage2_project(self, slices, out=None, stream=None):
        """Stage 2 + compounding + P-block sum-projection (ulm_rca_stage2_project).  slices: complex64 CUDA tensor
        [frame][compound = 0 output of beamform()]; returns complex64 [frame][planes_bytes_per_frame / 8]."""
        import torch
        if not self.stage2_block:
            raise ValueError("the plan was created without stage2_block")
        if not (slices.is_cuda and slices.dtype == torch.complex64 and slices.is_contiguous()
                and slices.device.index == self.device_index):
            raise ValueError("slices must be a contiguous complex64 CUDA tensor on the plan's device")
        n_frames = int(slices.shape[0])
        if n_frames and slices.numel() * 8 != n_frames * self.slices_bytes_per_frame:
            raise ValueError("slices have %d bytes per frame, plan expects %d" %
                             (slices.numel() * 8 // n_frames, self.slices_bytes_per_frame))
        if out is None:
            out = torch.empty((n_frames, self.planes_bytes_per_frame // 8), dtype=torch.complex64, device=slices.device)
        else:
            self._check_out(out, n_frames * self.planes_bytes_per_frame // 8)
        _check(load().ulm_rca_stage2_project(self._h, C.c_void_p(slices.data_ptr()), n_frames,
                                             C.c_void_p(out.data_ptr()), self._stream_ptr(stream)))
        return out

    def clutter_filter(self, slices, rank: int, out=None, want_eigenvalues: bool = False, want_covariance: bool = False,
                       stream=None):
        """Eigen-based clutter filter (ulm_rca_clutter_filter) on complex64 CUDA slices [frame][compound = 0 output].
        Returns the filtered slices, or (filtered, eigenvalues [n_events][32], covariance [n_events][n_t][n_t]) with the
        requested extras (None where not requested)."""
        import torch
        if not self.clutter_frames:
            raise ValueError("the plan was created without clutter_frames")
        if not (slices.is_cuda and slices.dtype == torch.complex64 and slices.is_contiguous()
                and slices.device.index == self.device_index and slices.dim() == 2
                and slices.shape[1] == self.slices_complex_per_frame):
            raise ValueError("slices must be a contiguous complex64 CUDA tensor [frame][%d] on the plan's device" % self.slices_complex_per_frame)
        n_t = int(slices.shape[0])
        if out is None:
            out = torch.empty_like(slices)
        else:
            self._check_out(out, slices.numel())
        lam = torch.empty((self.n_events, 32), dtype=torch.float32, device=slices.device) if want_eigenvalues else None
        cov = torch.empty((self.n_events, n_t, n_t), dtype=torch.complex64, device=slices.device) if want_covariance else None
        _check(load().ulm_rca_clutter_filter(self._h, C.c_void_p(slices.data_ptr()), n_t, int(rank), C.c_void_p(out.data_ptr()),
                                             C.c_void_p(lam.data_ptr()) if lam is not None else None,
                                             C.c_void_p(cov.data_ptr()) if cov is not None else None, self._stream_ptr(stream)))
        if want_eigenvalues or want_covariance:
            return out, lam, cov
        return out

    def localize(self, planes, sigma_lat_px: float, sigma_ax_px: float, threshold_rel: float, ncc_min: float, capacity: int = 64,
                 stream=None):
        """Separable 2-D NCC localization (ulm_rca_localize) on complex64 CUDA planes [frame][stage2 output].  Returns
        (loc float32 [frame][plane][capacity][4], count int32 [frame][plane]) as CUDA tensors."""
        import torch
        if not self.stage2_block:
            raise ValueError("the plan was created without stage2_block")
        if not (planes.is_cuda and planes.dtype == torch.complex64 and planes.is_contiguous() and planes.device.index == self.device_index
                and planes.dim() == 2 and planes.shape[1] * 8 == self.planes_bytes_per_frame):
            raise ValueError("planes must be a contiguous complex64 CUDA tensor [frame][%d]" % (self.planes_bytes_per_frame // 8))
        n = int(planes.shape[0])
        n_pl = self.n_planes_xz + self.n_planes_yz
        loc = torch.zeros((n, n_pl, int(capacity), 4), dtype=torch.float32, device=planes.device)
        count = torch.zeros((n, n_pl), dtype=torch.int32, device=planes.device)
        prm = LocalizeParams(float(sigma_lat_px), float(sigma_ax_px), float(threshold_rel), float(ncc_min), int(capacity))
        _check(load().ulm_rca_localize(self._h, C.c_void_p(planes.data_ptr()), n, C.byref(prm), C.c_void_p(loc.data_ptr()),
                                       C.c_void_p(count.data_ptr()), self._stream_ptr(stream)))
        return loc, count

    def motion_estimate(self, slices, ref_frame: int = 0, stream=None):
        """Fourier-domain NCC motion estimation (ulm_rca_motion_estimate).  Returns (motion float32 [frame][4] = dx, dy, dz
        in metres and mean NCC; per_event float32 [frame][event][4] = lateral px, axial px, NCC, 0) as CUDA tensors."""
        import torch
        if not self.motion_frames:
            raise ValueError("the plan was created without motion_frames")
        if not (slices.is_cuda and slices.dtype == torch.complex64 and slices.is_contiguous()
                and slices.device.index == self.device_index and slices.dim() == 2
                and slices.shape[1] == self.slices_complex_per_frame):
            raise ValueError("slices must be a contiguous complex64 CUDA tensor [frame][%d] on the plan's device" % self.slices_complex_per_frame)
        n = int(slices.shape[0])
        motion = torch.empty((n, 4), dtype=torch.float32, device=slices.device)
        per = torch.empty((n, self.n_events, 4), dtype=torch.float32, device=slices.device)
        _check(load().ulm_rca_motion_estimate(self._h, C.c_void_p(slices.data_ptr()), n, int(ref_frame), C.c_void_p(motion.data_ptr()),
                                              C.c_void_p(per.data_ptr()), self._stream_ptr(stream)))
        return motion, per

    def motion_timing(self) -> float:
        v = C.c_double()
        _check(load().ulm_rca_motion_timing(self._h, C.byref(v)))
        return float(v.value)

    def clutter_timing(self) -> tuple:
        """(split_ms, gram_ms, assemble_ms, eig_ms, project_ms) of the last clutter_filter() call."""
        v = (C.c_double * 5)()
        _check(load().ulm_rca_clutter_timing(self._h, v))
        return tuple(float(x) for x in v)

    def stage2_timing(self) -> tuple:
        """(groupsum_ms, project_ms) of the last batch of the last stage2_project() call."""
        a, b = C.c_double(), C.c_double()
        _check(load().ulm_rca_stage2_timing(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def beamform_host(self, channel: np.ndarray, out: Optional[np.ndarray] = None) -> np.ndarray:
        """Host-buffer entry (H2D + beamform + D2H + synchronise inside the library)."""
        channel = np.ascontiguousarray(channel, dtype=np.int16)
        n_frames = int(channel.shape[0])
        if n_frames and channel.nbytes != n_frames * self.channel_bytes_per_frame:
            raise ValueError("channel has the wrong size for this plan")
        if out is None:
            out = np.empty((n_frames, self.out_complex_per_frame), dtype=np.complex64)
        _check(load().ulm_rca_beamform_host(self._h, C.c_void_p(channel.ctypes.data), n_frames,
                                            C.c_void_p(out.ctypes.data)))
        return out

    def split(self, out_frame):
        """One frame of compound=1 output -> (P_xz [n_lat][n_ax], P_yz [n_lat][n_ax])."""
        nxz = self.grid_xz[0] * self.grid_xz[3]
        return (out_frame[:nxz].reshape(self.grid_xz[0], self.grid_xz[3]),
                out_frame[nxz:].reshape(self.grid_yz[0], self.grid_yz[3]))


def ring_probe(n_rx: int, pitch: float, angles: Sequence[float], c: float, fs: float, grid: tuple,
               t0: Optional[Sequence[float]] = None, t_start: float = 0.0) -> dict:
    """Host-only tile / window planning of the ring kernel for one aperture (ulm_rca_ring_probe)."""
    lib = load()
    aa, ap = _farr(list(angles))
    ta, tp = _farr(t0)
    g = Grid(*grid)
    nt, w = C.c_int32(), C.c_int32()
    _check(lib.ulm_rca_ring_probe(int(n_rx), float(pitch), ap, tp, len(angles), float(c), float(fs), float(t_start),
                                  C.byref(g), C.byref(nt), C.byref(w), None, None))
    dj = (C.c_int32 * (nt.value * n_rx))()
    wj = (C.c_int32 * (nt.value * n_rx))()
    _check(lib.ulm_rca_ring_probe(int(n_rx), float(pitch), ap, tp, len(angles), float(c), float(fs), float(t_start),
                                  C.byref(g), C.byref(nt), C.byref(w), dj, wj))
    return {"n_tiles": nt.value, "window": w.value,
            "dj": np.array(dj, dtype=np.int64).reshape(nt.value, n_rx),
            "wj": np.array(wj, dtype=np.int64).reshape(nt.value, n_rx)}


def fold_probe(angles: Sequence[float], c: float, fs: float, grid: tuple,
               t0: Optional[Sequence[float]] = None) -> list:
    """Host-only event folding of one aperture (ulm_rca_fold_probe): partner index, -1 (alone) or -2 (folded away)."""
    lib = load()
    aa, ap = _farr(list(angles))
    ta, tp = _farr(t0)
    g = Grid(*grid)
    out = (C.c_int32 * len(angles))()
    _check(lib.ulm_rca_fold_probe(ap, tp, len(angles), float(c), float(fs), C.byref(g), out))
    return [int(v) for v in out]


def fp32_peak_tflops(stream=None) -> float:
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    v = C.c_double()
    _check(load().ulm_rca_fp32_peak(C.byref(v), C.c_void_p(s.cuda_stream)))
    return float(v.value)

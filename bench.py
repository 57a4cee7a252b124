#!/usr/bin/env python
"""bench.py -- projection-beamformed frames/s on the 300-frame ensemble (BASELINE.json config 2).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2|3]

One "step" = one pass of the whole hot path (demodulation/staging pre-pass + DAS gather/compound +
projection write) over one 300-frame ensemble that is already resident in HBM.  Prints ONE JSON line
(contract in DESIGN.md "Measurement").  N > 1: one process per GPU (torchrun), every rank beamforms its
own ensemble (frames/ensembles are independent: no data-path collective), value = all frames / max time.
`--impl reference` times the fp64 CPU oracle (oracle/) on the host cores instead.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import synth  # noqa: E402
from helpers import rounded_kwargs  # noqa: E402

FLOP_PER_GATHER = 18.0           # algorithmic FP32 flop per (pixel, element, angle) term
NOMINAL_FP32_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12   # 148 SMs x 128 FP32 lanes x 2 flop x 1965 MHz
DISTINCT_FRAMES = (0, 100, 200, 299)   # frames of the moving scene rendered on the host and tiled


def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""
    REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
               0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag, self.max_mhz = index, [], set(), False, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        while not self.stop_flag and self.nv is not None:
            try:
                self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                mask = self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for bit, name in self.REASONS.items():
                    if mask & bit and name != "gpu_idle":
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.02)

    def result(self):
        self.stop_flag = True
        if self.is_alive():
            self.join(timeout=1.0)
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "samples": len(self.samples), "reasons": sorted(self.reasons)}


def whole_job(frames_per_rank: int, world: int, ms_local: float, all_reduce_max=None):
    """Whole-job throughput for independent per-rank ensembles: every rank beamforms frames_per_rank frames,
    the job takes the MAX over ranks of the device time (no data-path collective).  all_reduce_max(x) -> max over
    ranks of x (None for a single process).  Returns (frames/s, ms)."""
    ms = float(all_reduce_max(ms_local)) if (all_reduce_max is not None and world > 1) else float(ms_local)
    return world * frames_per_rank / (ms * 1e-3), ms


def prepass_roofline(cfg, info, n_frames, demod_ms):
    """HBM roofline of the staging pre-pass: algorithmic bytes = (2 B read + scratch bytes written) per touched
    (sample, frame) of the receive aperture of every event; peak = measured copy bandwidth (MEASURED_PEAKS.json)."""
    peak, src = 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md)"
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            peak, src = float(json.load(fh)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        pass
    rows = len(cfg.row_tx_angles) * cfg.n_cols + len(cfg.col_tx_angles) * cfg.n_rows
    fold = info["events_executed"] / float(len(cfg.row_tx_angles) + len(cfg.col_tx_angles))
    # every record of the receive apertures is read (2 B per sample); one scratch entry is written per FOLDED event
    byts = float(rows) * info["l_row"] * n_frames * (2 + fold * info["scratch_bytes_per_sample"])
    achieved = byts / (demod_ms * 1e-3) / 1e9
    return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "kernel": "demod_quad_kernel / demod_kernel", "algorithmic_bytes": byts, "peak_source": src}


def make_ensemble(cfg, torch, device):
    """Seeded synthetic ensemble in HBM: a few frames of the moving scene rendered on the host by synth/
    (the CPU echo simulator) and tiled over the n_frames-long buffer.  DAS cost does not depend on values."""
    distinct = [f for f in DISTINCT_FRAMES if f < cfg.n_frames] or [0]
    host = synth.render(cfg, distinct)
    dev = torch.from_numpy(host).to(device)
    idx = torch.arange(cfg.n_frames, device=device) % len(distinct)
    return dev[idx].contiguous(), host, distinct


def oracle_frames_per_s(cfg, host_frames, n_frames):
    """Time the fp64 oracle, as it stands, on n_frames frames (demodulation + both projections)."""
    import oracle
    p = oracle.OracleParams(**rounded_kwargs(cfg))
    reps = [host_frames[i % host_frames.shape[0]] for i in range(n_frames)]
    t0 = time.perf_counter()
    for fr in reps:
        oracle.beamform(p, fr[None])
    dt = time.perf_counter() - t0
    return n_frames / dt, dt, oracle.threads()


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2511_21647_b200 import Plan, build, fp32_peak_tflops

    rank, local_rank, world = dist_env()
    if world > 1:
        dist.init_process_group("nccl")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    build.build()
    cfg = synth.config(args.config)
    if args.per_angle:
        cfg = cfg.with_(compound=0)
    n_frames = cfg.n_frames
    channel, host_frames, distinct = make_ensemble(cfg, torch, device)
    gathers = cfg.gather_samples_per_frame() * n_frames

    plan = Plan(**rounded_kwargs(cfg), max_frames=n_frames)
    out = torch.empty((n_frames, plan.out_complex_per_frame), dtype=torch.complex64, device=device)
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        plan.beamform(channel, out=out)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    step_ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ev0.record(stream)
    for i in range(args.steps):
        plan.beamform(channel, out=out)
        step_ev[i].record(stream)
    ev1.record(stream)
    barrier()
    clocks = sampler.result()
    ms_total = ev0.elapsed_time(ev1)
    marks = [ev0] + step_ev
    per_step = sorted(marks[i].elapsed_time(marks[i + 1]) for i in range(args.steps))
    demod_ms, das_ms = plan.timing(min(args.steps, 64))
    info = plan.info()
    launches = info["launches_last_call"] * args.steps

    # end to end through the C-ABI host entry: pinned host buffers, H2D + kernels + D2H inside the timed region
    h_in = torch.empty(channel.shape, dtype=torch.int16, pin_memory=True)
    h_in.copy_(channel)
    h_out = torch.empty((n_frames, plan.out_complex_per_frame), dtype=torch.complex64, pin_memory=True)
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    plan.beamform_host(h_in.numpy(), out=h_out.numpy())           # allocates the library's staging once
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        plan.beamform_host(h_in.numpy(), out=h_out.numpy())
    e2e_s = time.perf_counter() - t0
    e2e_ms = torch.tensor([e2e_s * 1e3 / e2e_steps, ms_total / args.steps], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(e2e_ms, op=dist.ReduceOp.MAX)
    e2e_ms_step, ms_step = float(e2e_ms[0]), float(e2e_ms[1])

    fp32_probe = fp32_peak_tflops() if rank == 0 else None
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        fps1, dt1, cores = oracle_frames_per_s(cfg, host_frames, 1)
        n_more = int(np.clip(round(12.0 / max(dt1, 1e-3)), 1, 24))
        fps, dt, cores = oracle_frames_per_s(cfg, host_frames, n_more)
        cpu = {"value": fps, "unit": "frames/s", "cores": cores, "kind": "oracle",
               "sample": "%d frames of the %s workload (demodulation + both projections), %.1f s" % (n_more, cfg.name, dt)}
    plan.close()

    if rank == 0:
        # Roofline accounting: `gathers` = the pixel x element x angle terms of the definition;
        # the kernel executes fewer when transmit events fold (mirror angles about a centred reference slice are
        # added in the pre-pass and beamformed once).  The roofline fraction is taken on the EXECUTED terms -- the
        # conservative count; the unfolded (definition) count is reported beside it.
        n_events = len(cfg.row_tx_angles) + len(cfg.col_tx_angles)
        fold = info["events_executed"] / float(n_events)
        gathers_exec = gathers * fold
        achieved = FLOP_PER_GATHER * gathers_exec / (das_ms * 1e-3) / 1e12
        achieved_def = FLOP_PER_GATHER * gathers / (das_ms * 1e-3) / 1e12
        line = {
            "metric": "projection-beamformed frames/s (300-frame ensemble)" + (", one slice per transmit event (compound = 0)" if args.per_angle else ""),
            "value": whole_job(n_frames, world, ms_step)[0],
            "unit": "frames/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic: frames %s of the seeded moving scene rendered by synth/ (CPU echo "
            "simulator), tiled over the ensemble" % (list(distinct),),
            "config": {"workload": "BASELINE.json configs[%d] (%s): 128+128 RCA, 11+11 angles, %d frames, %dx%d px "
                       "per projection, %d samples @ %.0f MHz" % (args.config, cfg.name, n_frames, cfg.grid_xz[0],
                                                                   cfg.grid_xz[3], cfg.n_samples, cfg.fs / 1e6),
                       "frames": n_frames, "channel_bytes": int(channel.numel() * 2),
                       "l2_policy": "inputs (%.1f GB) larger than L2, no flush" % (channel.numel() * 2 / 1e9),
                       "parallelism": "independent ensembles per GPU, no collective", "plan": info},
            "gather_samples_per_s": world * gathers / (ms_step * 1e-3),
            "ms_per_step_min": per_step[0], "ms_per_step_median": per_step[len(per_step) // 2],
            "ensemble_ms": ms_step, "acquisition_ms": 1e3 * n_frames / cfg.frame_rate_hz,
            "kernels_ms": {"demod_stage": demod_ms, "das": das_ms},
            "roofline": {"bound": "alu", "achieved": achieved, "peak": NOMINAL_FP32_TFLOPS, "unit": "TFLOP/s",
                         "frac": achieved / NOMINAL_FP32_TFLOPS, "traffic": TRAFFIC_BYTES.get(args.config),
                         "kernel": "das_ring_kernel<12,4,%s,0>" % ("1" if info["precision"] == 2 else "0") if info["kernel"] == 2 else "das_generic_kernel",
                         "flop_per_gather_sample": FLOP_PER_GATHER, "gather_samples_per_launch": gathers_exec,
                         "gather_samples_of_the_definition": gathers, "events_executed_per_frame": info["events_executed"],
                         "events_per_frame": n_events, "frac_on_definition_count": achieved_def / NOMINAL_FP32_TFLOPS,
                         "peak_source": "derived: 148 SM x 128 lanes x 2 x 1965 MHz (DESIGN.md); FFMA probe measured "
                                        "%.1f TFLOP/s on this box" % fp32_probe,
                         "whole_step_frac": FLOP_PER_GATHER * gathers_exec / (ms_step * 1e-3) / 1e12 / NOMINAL_FP32_TFLOPS},
            "roofline_prepass": prepass_roofline(cfg, info, n_frames, demod_ms),
            "cpu_baseline": cpu, "clocks": clocks,
            "e2e": {"value": world * n_frames / (e2e_ms_step * 1e-3), "unit": "frames/s",
                    "h2d_bytes_per_step": int(info["host_upload_bytes_per_frame"]) * n_frames,
                    "host_buffer_bytes": int(channel.numel() * 2), "d2h_bytes_per_step": int(out.numel() * 8),
                    "ms_per_step": e2e_ms_step, "steps": e2e_steps},
            "gpu_launches": int(launches),
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel per launch, from the ncu --set full
# capture summarised under profiles/ (None until captured for that config)
TRAFFIC_BYTES = {2: 3.677742e9 + 0.195292e9,      # profiles/r01_v7_ncu.md (das_ring_kernel<12,4,0,0>, one launch)
                 3: 7.129134e9 + 0.556273e9}      # profiles/r01_v7_cfg3.md


def run_volume(args):
    """Config 4, the paper's conventional comparator: cfg 1's data beamformed as a full
    180 x 180 x 164 volume by unpack_frame_kernel + das_volume_kernel (one frame); reported as volumes/s next to the
    projection path's frames/s."""
    import torch
    from paper_2511_21647_b200 import Plan, build
    torch.cuda.set_device(0)
    build.build()
    cfg = synth.config(4)
    host = synth.render(cfg)
    ch = torch.from_numpy(host).cuda()
    gathers = cfg.gather_samples_per_frame()
    with Plan(**rounded_kwargs(cfg), build_volume=True, max_frames=1) as plan:
        out = plan.beamform_volume(ch)
        for _ in range(max(args.warmup, 3)):
            plan.beamform_volume(ch, out=out)
        torch.cuda.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for _ in range(args.steps):
            plan.beamform_volume(ch, out=out)
        ev1.record()
        torch.cuda.synchronize()
        ms = ev0.elapsed_time(ev1) / args.steps
        launches = int(plan.info()["launches_last_call"])
        # the projection path on the same frame, for the speed ratio
        proj = plan.beamform(ch)
        torch.cuda.synchronize()
        ev0.record()
        for _ in range(args.steps):
            plan.beamform(ch, out=proj)
        ev1.record()
        torch.cuda.synchronize()
        ms_proj = ev0.elapsed_time(ev1) / args.steps
    achieved = FLOP_PER_GATHER * gathers / (ms * 1e-3) / 1e12
    print(json.dumps({
        "metric": "full-3D DAS volumes/s (config 4, conventional comparator)", "value": 1e3 / ms, "unit": "volumes/s",
        "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic: config 1 frame rendered by synth/",
        "config": {"workload": "BASELINE.json configs[4]: 180x180x164 voxels, 11+11 angles, 128+128 RCA, 1 frame"},
        "gather_samples_per_s": gathers / (ms * 1e-3),
        "projection_path_ms_same_frame": ms_proj, "volume_over_projection_time": ms / ms_proj,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": NOMINAL_FP32_TFLOPS, "unit": "TFLOP/s",
                     "frac": achieved / NOMINAL_FP32_TFLOPS, "traffic": 19.985152e6 + 0.501760e6, "kernel": "das_volume_kernel<4,0>"},
        "gpu_launches": launches * args.steps}))


def run_reference(args):
    """Reference arm of this tier: the fp64 oracle, as it stands, on the host cores (rank 0 only).
    Each step beamforms `ref_frames` frames of the same workload (a bounded sample of the ensemble)."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    import oracle
    cfg = synth.config(args.config)
    oracle.build()
    distinct = [f for f in DISTINCT_FRAMES if f < cfg.n_frames] or [0]
    host = synth.render(cfg, distinct[:max(1, min(len(distinct), args.ref_frames))])
    p = oracle.OracleParams(**rounded_kwargs(cfg))

    def step(i):
        for r in range(args.ref_frames):
            oracle.beamform(p, host[(i + r) % host.shape[0]][None])

    for i in range(args.warmup):
        step(i)
    t0 = time.perf_counter()
    for i in range(args.steps):
        step(i)
    dt = time.perf_counter() - t0
    fps = args.steps * args.ref_frames / dt
    line = {"impl": "reference", "metric": "projection-beamformed frames/s (300-frame ensemble)", "value": fps,
            "unit": "frames/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic: frames %s of the seeded moving scene rendered by synth/" % (distinct,),
            "config": {"workload": "BASELINE.json configs[%d] (%s), %d frame(s) per step" % (args.config, cfg.name, args.ref_frames)},
            "cpu_baseline": {"value": fps, "unit": "frames/s", "cores": oracle.threads(), "kind": "oracle",
                             "sample": "%d frame(s) per step of the %s workload (demodulation + both projections)" % (args.ref_frames, cfg.name)},
            "e2e": {"value": fps, "unit": "frames/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=[2, 3, 4])
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--ref-frames", type=int, default=1)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--per-angle", action="store_true",
                    help="compound = 0: one slice per transmit event (the paper's S_k) instead of the compounded "
                         "projections -- a secondary figure, not the BASELINE metric")
    args = ap.parse_args()
    if args.steps < 1:
        ap.error("--steps must be >= 1")
    _, _, world = dist_env()
    if world != max(1, args.gpus):
        if world == 1 and args.gpus > 1:
            sys.stderr.write("bench.py: --gpus %d needs torchrun with --nproc-per-node %d; running 1 GPU\n" % (args.gpus, args.gpus))
    if args.impl == "reference":
        run_reference(args)
    elif args.config == 4:
        run_volume(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

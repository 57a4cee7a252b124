#!/usr/bin/env python
"""bench.py -- projection-beamformed frames/s on the 300-frame ensemble (BASELINE.json config 2).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2|3|4]

One "step" = one pass of the whole hot path (demodulation/staging pre-pass + DAS gather/compound +
projection write) over one 300-frame ensemble that is already resident in HBM.  Prints ONE JSON line
(contract in DESIGN.md "Measurement").  N > 1: one process per GPU, every rank beamforms its own ensemble
(frames/ensembles are independent: no data-path collective), value = all frames / max time; when the script is
started without a launcher (WORLD_SIZE unset) it starts the N ranks itself through torch.distributed.run and fails
if fewer than N GPUs are visible.
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


def measured_traffic(config_index: int, precision: int):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, read from the summary of the
    `ncu --set full` capture under profiles/ (profiles/r02_traffic.json; its .md names the commands).  None when no
    capture of that (config, precision) exists."""
    try:
        with open(os.path.join(ROOT, "profiles", "r02_traffic.json")) as fh:
            rec = json.load(fh)["das_ring_kernel"]["cfg%d_precision%d" % (config_index, precision)]
        return float(rec["dram_bytes_read"]) + float(rec["dram_bytes_write"])
    except Exception:
        return None


def capture_traffic(name: str):
    """The same figure for the dominant kernel of another workload (profiles/r02_traffic.json, section "captures")."""
    try:
        with open(os.path.join(ROOT, "profiles", "r02_traffic.json")) as fh:
            rec = json.load(fh)["captures"][name]
        return float(rec["dram_bytes_read"]) + float(rec["dram_bytes_write"])
    except Exception:
        return None


DTYPE_OF_PRECISION = {1: "f32 accumulate; staged IQ: fp24 mid + fp16 difference, fp16 weight (precision=1, compact-fast)",
                      2: "f32 (staged IQ, interpolation and accumulation all fp32; precision=2)",
                      3: "f32 accumulate; staged IQ: fp24 mid + fp16 difference, two-term fp16 weight (precision=3, compact)"}


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
    """Time the fp64 oracle, as it stands, on n_frames frames (demodulation + both projections).  Also returns its
    output for each distinct host frame it saw ({index into host_frames: complex128 frame})."""
    import oracle
    p = oracle.OracleParams(**rounded_kwargs(cfg))
    outs = {}
    t0 = time.perf_counter()
    for i in range(n_frames):
        d = i % host_frames.shape[0]
        outs[d] = oracle.beamform(p, host_frames[d][None])[0]
    dt = time.perf_counter() - t0
    return n_frames / dt, dt, oracle.threads(), outs


def time_arm(torch, plan, channel, out, steps, warmup, barrier, local_rank, sample_clocks=False):
    """W untimed + K timed whole-ensemble calls of ulm_rca_beamform on torch's current stream, CUDA events on that
    stream, barrier + synchronize on both sides.  Returns a dict of timings."""
    stream = torch.cuda.current_stream()
    for _ in range(warmup):
        plan.beamform(channel, out=out)
    barrier()
    sampler = ClockSampler(local_rank) if sample_clocks else None
    if sampler:
        sampler.start()
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    marks[0].record(stream)
    for i in range(steps):
        plan.beamform(channel, out=out)
        marks[i + 1].record(stream)
    barrier()
    clocks = sampler.result() if sampler else None
    per_step = sorted(marks[i].elapsed_time(marks[i + 1]) for i in range(steps))
    demod_ms, das_ms = plan.timing(min(steps, 64))
    info = plan.info()
    return {"ms_step": marks[0].elapsed_time(marks[steps]) / steps, "per_step": per_step, "demod_ms": demod_ms,
            "das_ms": das_ms, "info": info, "launches": info["launches_last_call"] * steps, "clocks": clocks}


def das_roofline(cfg, args, arm, gathers, fp32_probe, world_ms=None):
    """ALU roofline of the DAS kernel: achieved = 18 flop x EXECUTED gather-samples / the
    kernel's mean duration (CUDA events the library records on the launching stream); peak = derived FP32 peak,
    with the in-run FFMA probe beside it."""
    info = arm["info"]
    n_events = len(cfg.row_tx_angles) + len(cfg.col_tx_angles)
    fold = info["events_executed"] / float(n_events)
    gathers_exec = gathers * fold
    achieved = FLOP_PER_GATHER * gathers_exec / (arm["das_ms"] * 1e-3) / 1e12
    achieved_def = FLOP_PER_GATHER * gathers / (arm["das_ms"] * 1e-3) / 1e12
    ms_step = world_ms if world_ms is not None else arm["ms_step"]
    # the kernel's own shared-memory floor: bytes of scratch entries gathered per executed term at 128 B/clk/SM
    smem_floor_ms = gathers_exec * info["scratch_bytes_per_sample"] / (148 * 128 * 1.965e9) * 1e3
    return {"bound": "alu", "achieved": achieved, "peak": NOMINAL_FP32_TFLOPS, "unit": "TFLOP/s",
            "frac": achieved / NOMINAL_FP32_TFLOPS,
            "peak_measured": fp32_probe, "frac_of_measured": (achieved / fp32_probe) if fp32_probe else None,
            "traffic": measured_traffic(args.config, info["precision"]) if not args.per_angle else None,
            # compact entries, more than 12 frames: work items of two frame groups, 2 pixel rows (template <F, PX, D32, APOD, W2, DUAL>)
            "kernel": (("das_ring_kernel<12,4,1,0,0,0>" if info["precision"] == 2 else
                        "das_ring_kernel<12,2,0,0,%d,1> (+ <12,4,0,0,%d,0> for an odd last frame group)" % ((info["precision"] == 3,) * 2))
                       if info["kernel"] == 2 else "das_generic_kernel"),
            "precision": info["precision"], "kernel_ms": arm["das_ms"], "prepass_ms": arm["demod_ms"],
            "flop_per_gather_sample": FLOP_PER_GATHER, "gather_samples_per_launch": gathers_exec,
            "gather_samples_of_the_definition": gathers, "events_executed_per_frame": info["events_executed"],
            "events_per_frame": n_events, "frac_on_definition_count": achieved_def / NOMINAL_FP32_TFLOPS,
            "peak_source": "derived: 148 SM x 128 lanes x 2 x 1965 MHz (DESIGN.md section 8); peak_measured = the "
                           "library's register-only FFMA probe run in this process",
            "whole_step_frac": FLOP_PER_GATHER * gathers_exec / (ms_step * 1e-3) / 1e12 / NOMINAL_FP32_TFLOPS,
            "smem_floor_ms": smem_floor_ms, "frac_of_smem_floor": smem_floor_ms / arm["das_ms"]}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2511_21647_b200 import Plan, build, fp32_peak_tflops

    rank, local_rank, world = dist_env()
    if world > 1:
        dist.init_process_group("nccl")
    if torch.cuda.device_count() <= local_rank:
        sys.stderr.write("bench.py: rank %d needs cuda:%d but only %d device(s) are visible\n" % (rank, local_rank, torch.cuda.device_count()))
        sys.exit(2)
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    build.build()
    cfg = synth.config(args.config)
    if args.per_angle:
        cfg = cfg.with_(compound=0)
    n_frames = cfg.n_frames
    channel, host_frames, distinct = make_ensemble(cfg, torch, device)
    gathers = cfg.gather_samples_per_frame() * n_frames
    warmup = max(args.warmup, 3)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def all_max(x):
        v = torch.tensor([x], dtype=torch.float64, device=device)
        dist.all_reduce(v, op=dist.ReduceOp.MAX)
        return float(v[0])

    plan = Plan(**rounded_kwargs(cfg), max_frames=n_frames, precision=args.precision)
    out = torch.empty((n_frames, plan.out_complex_per_frame), dtype=torch.complex64, device=device)
    arm = time_arm(torch, plan, channel, out, args.steps, warmup, barrier, local_rank, sample_clocks=True)
    info = arm["info"]
    got_default = out[:len(distinct)].cpu().numpy()

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
    e2e_ms_step = (time.perf_counter() - t0) * 1e3 / e2e_steps
    ms_step = arm["ms_step"]
    if world > 1:
        e2e_ms_step, ms_step = all_max(e2e_ms_step), all_max(ms_step)
    plan.close()
    del h_in, h_out

    # the other scratch formats on the same workload (rank 0 of a single-GPU run only): the driver-run record shows
    # the precision / speed trade next to the default arm
    arms = {}
    if rank == 0 and world == 1 and not args.no_arms and not args.per_angle:
        for prec in (1, 2, 3):
            if prec == info["precision"]:
                continue
            with Plan(**rounded_kwargs(cfg), max_frames=n_frames, precision=prec) as p2:
                a = time_arm(torch, p2, channel, out, max(3, min(args.steps, 6)), 3, barrier, local_rank)
                a["got"] = out[:len(distinct)].cpu().numpy()
                arms[prec] = a

    fp32_probe = fp32_peak_tflops() if rank == 0 else None
    cpu, parity = None, {}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        fps1, dt1, cores, _ = oracle_frames_per_s(cfg, host_frames, 1)
        n_more = int(np.clip(round(12.0 / max(dt1, 1e-3)), len(distinct), 24))
        fps, dt, cores, refs = oracle_frames_per_s(cfg, host_frames, n_more)
        cpu = {"value": fps, "unit": "frames/s", "cores": cores, "kind": "oracle",
               "sample": "%d frames of the %s workload (demodulation + both projections), %.1f s" % (n_more, cfg.name, dt)}

        def worst(got):
            return max(float(np.abs(got[d] - refs[d]).max() / np.abs(refs[d]).max()) for d in refs)

        parity[info["precision"]] = worst(got_default)
        for prec, a in arms.items():
            parity[prec] = worst(a["got"])

    if rank == 0:
        roof = das_roofline(cfg, args, arm, gathers, fp32_probe, world_ms=ms_step)
        roof["parity_max_rel_err_vs_oracle"] = parity.get(info["precision"])
        line = {
            "metric": "projection-beamformed frames/s (300-frame ensemble)" + (", one slice per transmit event (compound = 0)" if args.per_angle else ""),
            "value": world * n_frames / (ms_step * 1e-3),
            "unit": "frames/s", "n_gpus": world, "steps": args.steps, "warmup": warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": DTYPE_OF_PRECISION[info["precision"]],
            "data": "synthetic: frames %s of the seeded moving scene rendered by synth/ (CPU echo "
            "simulator), tiled over the ensemble" % (list(distinct),),
            "config": {"workload": "BASELINE.json configs[%d] (%s): 128+128 RCA, 11+11 angles, %d frames, %dx%d px "
                       "per projection, %d samples @ %.0f MHz" % (args.config, cfg.name, n_frames, cfg.grid_xz[0],
                                                                   cfg.grid_xz[3], cfg.n_samples, cfg.fs / 1e6),
                       "frames": n_frames, "channel_bytes": int(channel.numel() * 2),
                       "l2_policy": "inputs (%.1f GB) larger than L2, no flush" % (channel.numel() * 2 / 1e9),
                       "parallelism": "independent ensembles per GPU, no collective",
                       "precision_requested": args.precision, "plan": info},
            "gather_samples_per_s": world * gathers / (ms_step * 1e-3),
            "ms_per_step_min": arm["per_step"][0], "ms_per_step_median": arm["per_step"][len(arm["per_step"]) // 2],
            "ensemble_ms": ms_step, "acquisition_ms": 1e3 * n_frames / cfg.frame_rate_hz,
            "kernels_ms": {"demod_stage": arm["demod_ms"], "das": arm["das_ms"]},
            "roofline": roof,
            "roofline_prepass": prepass_roofline(cfg, info, n_frames, arm["demod_ms"]),
            "cpu_baseline": cpu, "clocks": arm["clocks"],
            "e2e": {"value": world * n_frames / (e2e_ms_step * 1e-3), "unit": "frames/s",
                    "h2d_bytes_per_step": int(info["host_upload_bytes_per_frame"]) * n_frames,
                    "host_buffer_bytes": int(channel.numel() * 2), "d2h_bytes_per_step": int(out.numel() * 8),
                    "ms_per_step": e2e_ms_step, "steps": e2e_steps},
            "gpu_launches": int(arm["launches"]),
        }
        names = {1: "roofline_compact_fast", 2: "roofline_full", 3: "roofline_compact"}
        for prec, a in arms.items():
            r = das_roofline(cfg, args, a, gathers, fp32_probe)
            r["parity_max_rel_err_vs_oracle"] = parity.get(prec)
            r["frames_per_s"] = n_frames / (a["ms_step"] * 1e-3)
            r["steps"] = len(a["per_step"])
            line[names[prec]] = r
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        return 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md)"


def run_stage2(args):
    """NEXT-1: Stage-2 extrapolation + compounding over 2K + P = 8 sum-projection (PAPER.md:45, 79, 93,
    117) on the per-event slices of a 300-frame ensemble of config 2's shape: 22 slices of 180 x 164 px per frame ->
    23 + 23 projected planes per frame.  One step = ulm_rca_stage2_project over the whole ensemble, slices resident in
    HBM (1.56 GB in, 3.26 GB out: larger than L2)."""
    import torch
    from paper_2511_21647_b200 import Plan, build, fp32_peak_tflops
    torch.cuda.set_device(0)
    build.build()
    cfg = synth.config(2).with_(compound=0)
    n_frames, block = cfg.n_frames, 8
    kw = rounded_kwargs(cfg)
    per_frame = len(cfg.row_tx_angles) * cfg.grid_xz[0] * cfg.grid_xz[3] + len(cfg.col_tx_angles) * cfg.grid_yz[0] * cfg.grid_yz[3]
    n_distinct = 3
    distinct = synth.random_complex((n_distinct, per_frame), 21, amplitude=50.0)
    idx = torch.arange(n_frames, device="cuda") % n_distinct
    slices = torch.from_numpy(distinct).cuda()[idx].contiguous()
    warmup = max(args.warmup, 3)
    with Plan(**kw, stage2_block=block, max_frames=n_frames) as plan:
        out = plan.stage2_project(slices)
        for _ in range(warmup):
            plan.stage2_project(slices, out=out)
        torch.cuda.synchronize()
        sampler = ClockSampler(0)
        sampler.start()
        stream = torch.cuda.current_stream()
        marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
        gs_ms = pj_ms = 0.0
        marks[0].record(stream)
        for i in range(args.steps):
            plan.stage2_project(slices, out=out)
            marks[i + 1].record(stream)
        torch.cuda.synchronize()
        clocks = sampler.result()
        ms = marks[0].elapsed_time(marks[args.steps]) / args.steps
        gs_ms, pj_ms = plan.stage2_timing()
        info = plan.info()
        n_g = (plan.n_planes_xz, plan.n_planes_yz)
        got = out[:n_distinct].cpu().numpy()
        # end to end: pinned host slices -> device -> planes -> pinned host
        h_in = torch.empty(slices.shape, dtype=torch.complex64, pin_memory=True)
        h_in.copy_(slices)
        h_out = torch.empty(out.shape, dtype=torch.complex64, pin_memory=True)
        d_in = torch.empty_like(slices)
        t0 = time.perf_counter()
        for _ in range(2):
            d_in.copy_(h_in, non_blocking=True)
            plan.stage2_project(d_in, out=out)
            h_out.copy_(out, non_blocking=True)
            torch.cuda.synchronize()
        e2e_ms = (time.perf_counter() - t0) * 1e3 / 2
    fp32_probe = fp32_peak_tflops()
    # work: definition = every (voxel, event) term: linear interpolation (6 flop) + carrier rotation-accumulate (8) +
    # block sum (2); executed = complex multiply-adds of the factored form, 8 flop each
    nx, ny, nz = cfg.grid_xz[0], cfg.grid_yz[0], cfg.grid_xz[3]
    kr, kc = len(cfg.row_tx_angles), len(cfg.col_tx_angles)
    terms_def = float(nx) * ny * nz * (kr + kc) * 2 * n_frames          # each voxel term feeds both plane stacks
    cmac = float(n_frames) * nz * (n_g[0] * nx * (kr * info["stage2_taps"] + kc * 2) + n_g[1] * ny * (kc * info["stage2_taps"] + kr * 2))
    flop_exec, flop_def = 8.0 * cmac, 16.0 * terms_def
    byts = float(slices.numel() + out.numel()) * 8
    peak_hbm, hbm_src = hbm_peak()
    t_alu, t_hbm = flop_exec / (NOMINAL_FP32_TFLOPS * 1e12) * 1e3, byts / (peak_hbm * 1e9) * 1e3
    cpu = None
    if not args.no_cpu_baseline:
        import oracle
        from oracle import stage2
        p = oracle.OracleParams(**kw)
        t0 = time.perf_counter()
        ref = stage2.stage2_planes(p, distinct[:2].astype(np.complex128), block)
        dt = time.perf_counter() - t0
        parity = max(float(np.abs(got[i] - ref[i]).max() / np.abs(ref[i]).max()) for i in range(2))
        cpu = {"value": 2 / dt, "unit": "frames/s", "cores": 1, "kind": "oracle",
               "sample": "2 frames of the same slices (oracle/stage2.py, numpy fp64, single thread), %.1f s" % dt,
               "parity_max_rel_err_vs_oracle": parity}
    print(json.dumps({
        "metric": "Stage-2 + compounding + P=8 sum-projected frames/s (300-frame ensemble)", "value": n_frames / (ms * 1e-3),
        "unit": "frames/s", "n_gpus": 1, "steps": args.steps, "warmup": warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32 complex (taps built in fp64 on the host)",
        "data": "synthetic: 3 seeded random complex slice sets (synth.random_complex) tiled over 300 frames",
        "config": {"workload": "SURVEY 8(f) NEXT-1 on BASELINE configs[2] shapes: 300 frames x 22 slices of %dx%d px -> %d+%d "
                               "planes (P = %d)" % (nx, nz, n_g[0], n_g[1], block),
                   "l2_policy": "inputs + outputs (%.1f GB) larger than L2, no flush" % (byts / 1e9), "plan": info},
        "kernels_ms": {"groupsum": gs_ms, "project": pj_ms},
        "roofline": {"bound": "alu", "achieved": flop_exec / (pj_ms * 1e-3) / 1e12, "peak": NOMINAL_FP32_TFLOPS, "unit": "TFLOP/s",
                     "frac": flop_exec / (pj_ms * 1e-3) / 1e12 / NOMINAL_FP32_TFLOPS, "peak_measured": fp32_probe,
                     "frac_of_measured": flop_exec / (pj_ms * 1e-3) / 1e12 / fp32_probe, "traffic": capture_traffic("r02_stage2"),
                     "kernel": "stage2_project_kernel<%d>" % info["stage2_taps"], "kernel_ms": pj_ms,
                     "executed_complex_macs": cmac, "flop_executed": flop_exec, "flop_of_the_definition": flop_def,
                     "frac_on_definition_count": flop_def / (pj_ms * 1e-3) / 1e12 / NOMINAL_FP32_TFLOPS,
                     "alu_bound_ms": t_alu, "hbm_bound_ms": t_hbm, "algorithmic_bytes": byts,
                     "hbm_frac_whole_step": byts / (ms * 1e-3) / 1e9 / peak_hbm, "hbm_peak_source": hbm_src},
        "cpu_baseline": cpu, "clocks": clocks,
        "e2e": {"value": n_frames / (e2e_ms * 1e-3), "unit": "frames/s", "h2d_bytes_per_step": int(slices.numel() * 8),
                "d2h_bytes_per_step": int(out.numel() * 8), "ms_per_step": e2e_ms, "steps": 2},
        "gpu_launches": int(info["launches_last_call"]) * args.steps}))


def run_clutter(args):
    """NEXT-2: eigen-based clutter filter on the per-event slice stacks of a 300-frame
    ensemble of config 2's shape: 22 stacks of 300 x 29 520 complex values; one step = ulm_rca_clutter_filter (bf16 split,
    tcgen05 Gram kernel, assembly, eigen-subspace, projection), slices resident in HBM (1.56 GB > L2)."""
    import torch
    from paper_2511_21647_b200 import Plan, build
    torch.cuda.set_device(0)
    build.build()
    cfg = synth.config(2).with_(compound=0)
    n_t, rank = cfg.n_frames, 4
    kw = rounded_kwargs(cfg)
    n_pix = [cfg.grid_xz[0] * cfg.grid_xz[3]] * len(cfg.row_tx_angles) + [cfg.grid_yz[0] * cfg.grid_yz[3]] * len(cfg.col_tx_angles)
    x = synth.clutter_ensemble(n_t, n_pix, seed=22, tissue_rank=rank)
    d_x = torch.from_numpy(x).cuda()
    warmup = max(args.warmup, 3)
    with Plan(**kw, clutter_frames=n_t) as plan:
        out = plan.clutter_filter(d_x, rank)
        for _ in range(warmup):
            plan.clutter_filter(d_x, rank, out=out)
        torch.cuda.synchronize()
        sampler = ClockSampler(0)
        sampler.start()
        stream = torch.cuda.current_stream()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        for _ in range(args.steps):
            plan.clutter_filter(d_x, rank, out=out)
        ev1.record(stream)
        torch.cuda.synchronize()
        clocks = sampler.result()
        ms = ev0.elapsed_time(ev1) / args.steps
        k_ms = dict(zip(("split", "gram", "assemble", "eig", "project"), plan.clutter_timing()))
        info = plan.info()
        h_in = torch.empty(d_x.shape, dtype=torch.complex64, pin_memory=True)
        h_in.copy_(d_x)
        h_out = torch.empty(d_x.shape, dtype=torch.complex64, pin_memory=True)
        d_in = torch.empty_like(d_x)
        t0 = time.perf_counter()
        for _ in range(2):
            d_in.copy_(h_in, non_blocking=True)
            plan.clutter_filter(d_in, rank, out=out)
            h_out.copy_(out, non_blocking=True)
            torch.cuda.synchronize()
        e2e_ms = (time.perf_counter() - t0) * 1e3 / 2
        got = out[:, :n_pix[0]].cpu().numpy()
    # tensor-core roofline of the Gram kernel: algorithmic = 8 flop per complex multiply-add of C = I^H I (full, not the
    # Hermitian half); executed = the bf16 x 3 real products over the upper-triangular 128 x 128 tiles of the padded Gram
    n_ev = len(n_pix)
    flop_alg = 8.0 * n_t * n_t * float(sum(n_pix))
    nr = 2 * ((n_t + 63) // 64 * 64)
    tiles = (nr // 128) * (nr // 128 + 1) // 2
    flop_exec = 3 * 2.0 * tiles * 128 * 128 * ((max(n_pix) + 63) // 64 * 64) * n_ev
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            peak, src = float(json.load(fh)["bf16_tflops"]), "MEASURED_PEAKS.json bf16_tflops (burst: the kernel is timed alone by CUDA events)"
    except Exception:
        peak, src = 1590.0, "fallback 1.59 PFLOP/s (B200_PROFILING.md)"
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import clutter
        t0 = time.perf_counter()
        ref, lam, _ = clutter.clutter_filter_stack(x[:, :n_pix[0]].astype(np.complex128), rank)
        dt = time.perf_counter() - t0
        cpu = {"value": n_t / (dt * n_ev), "unit": "frames/s", "cores": int(os.cpu_count() or 1), "kind": "oracle",
               "sample": "1 of the %d slice stacks (oracle/clutter.py, numpy fp64 + LAPACK threads), %.1f s; scaled to %d stacks" % (n_ev, dt, n_ev),
               "parity_max_err_over_max_input": float(np.abs(got - ref).max() / np.abs(x).max())}
    print(json.dumps({
        "metric": "clutter-filtered frames/s (300-frame ensemble, 22 slice stacks)", "value": n_t / (ms * 1e-3), "unit": "frames/s",
        "n_gpus": 1, "steps": args.steps, "warmup": warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "bf16 x 3 split operands, fp32 accumulate (covariance); fp32 (eigen-subspace, projection)",
        "data": "synthetic: synth.clutter_ensemble (rank-4 tissue 30 dB above sparse bubbles + noise), seed 22",
        "config": {"workload": "SURVEY 8(f) NEXT-2 on BASELINE configs[2] shapes: 22 stacks of 300 frames x 29520 px, clutter rank 4",
                   "l2_policy": "inputs (%.2f GB) larger than L2, no flush" % (d_x.numel() * 8 / 1e9), "plan": info},
        "kernels_ms": k_ms,
        "roofline": {"bound": "tensor", "achieved": flop_alg / (k_ms["gram"] * 1e-3) / 1e12, "peak": peak, "unit": "TFLOP/s",
                     "frac": flop_alg / (k_ms["gram"] * 1e-3) / 1e12 / peak, "traffic": capture_traffic("r02_clutter"), "kernel": "clutter_gram_kernel",
                     "kernel_ms": k_ms["gram"], "flop_algorithmic": flop_alg, "flop_executed": flop_exec,
                     "achieved_executed": flop_exec / (k_ms["gram"] * 1e-3) / 1e12,
                     "frac_executed": flop_exec / (k_ms["gram"] * 1e-3) / 1e12 / peak, "peak_source": src},
        "cpu_baseline": cpu, "clocks": clocks,
        "e2e": {"value": n_t / (e2e_ms * 1e-3), "unit": "frames/s", "h2d_bytes_per_step": int(d_x.numel() * 8),
                "d2h_bytes_per_step": int(d_x.numel() * 8), "ms_per_step": e2e_ms, "steps": 2},
        "gpu_launches": int(info["launches_last_call"]) * args.steps}))


def run_motion(args):
    """NEXT-3: Fourier-domain NCC rigid motion estimation on the per-event slices of a
    300-frame ensemble of config 2's shape (22 slices of 180 x 164 px per frame, 256 x 256 transforms), every frame
    against frame 0; one step = ulm_rca_motion_estimate over the whole ensemble, slices resident in HBM."""
    import torch
    from paper_2511_21647_b200 import Plan, build
    torch.cuda.set_device(0)
    build.build()
    cfg = synth.config(2).with_(compound=0)
    kw = rounded_kwargs(cfg)
    n_frames = cfg.n_frames
    shapes = [(cfg.grid_xz[0], cfg.grid_xz[3])] * len(cfg.row_tx_angles) + [(cfg.grid_yz[0], cfg.grid_yz[3])] * len(cfg.col_tx_angles)
    shifts = [(0.0, 0.0), (0.8, -0.6), (-1.4, 0.35), (2.6, 1.2)]
    distinct = synth.moving_speckle(4, shapes, shifts, seed=2)
    idx = torch.arange(n_frames, device="cuda") % 4
    d = torch.from_numpy(distinct).cuda()[idx].contiguous()
    warmup = max(args.warmup, 3)
    with Plan(**kw, motion_frames=n_frames) as plan:
        for _ in range(warmup):
            mot, per = plan.motion_estimate(d, 0)
        torch.cuda.synchronize()
        sampler = ClockSampler(0)
        sampler.start()
        stream = torch.cuda.current_stream()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        for _ in range(args.steps):
            mot, per = plan.motion_estimate(d, 0)
        ev1.record(stream)
        torch.cuda.synchronize()
        clocks = sampler.result()
        ms = ev0.elapsed_time(ev1) / args.steps
        k_ms = plan.motion_timing()
        info = plan.info()
        h_in = torch.empty(d.shape, dtype=torch.complex64, pin_memory=True)
        h_in.copy_(d)
        d_in = torch.empty_like(d)
        t0 = time.perf_counter()
        for _ in range(2):
            d_in.copy_(h_in, non_blocking=True)
            m2, _ = plan.motion_estimate(d_in, 0)
            m_host = m2.cpu()
        e2e_ms = (time.perf_counter() - t0) * 1e3 / 2
        per = per.cpu().numpy()
    # HBM roofline: bytes the six kernels must move (slices read twice: the statistics pass and the forward
    # transform; T1 and T2 written and read once each per PACKED image = two frames) vs the minimum (slices read once);
    # flops: 2 two-dimensional 256 x 256 transforms per packed image (forward, inverse), 5 N log2 N each
    n_img = ((n_frames + 1) // 2) * len(shapes)
    fft_flop = 2 * 5.0 * (256 * 256) * 16 * n_img
    bytes_min = float(d.numel() * 8)
    bytes_moved = float(d.numel() * 8 * 2 + n_img * (256 * 192 * 8 * 2 + 256 * 256 * 8 * 2))
    peak_hbm, hbm_src = hbm_peak()
    cpu = None
    if not args.no_cpu_baseline:
        import oracle
        from oracle import motion
        t0 = time.perf_counter()
        per_ref, _ = motion.estimate(oracle.OracleParams(**kw), distinct.astype(np.complex128), 0)
        dt = time.perf_counter() - t0
        cpu = {"value": 4 / dt, "unit": "frames/s", "cores": 1, "kind": "oracle",
               "sample": "the 4 distinct frames x 22 slices (oracle/motion.py, numpy.fft fp64), %.1f s" % dt,
               "parity_max_shift_err_px": float(np.abs(per[:4, :, :2] - per_ref[:, :, :2]).max())}
    print(json.dumps({
        "metric": "motion-estimated frames/s (300-frame ensemble, 22 slices per frame)", "value": n_frames / (ms * 1e-3), "unit": "frames/s",
        "n_gpus": 1, "steps": args.steps, "warmup": warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32 (hand-written warp FFTs in registers, two frames per complex transform)",
        "data": "synthetic: synth.moving_speckle, 4 distinct frames with programmed sub-pixel shifts tiled over 300 frames",
        "config": {"workload": "SURVEY 8(f) NEXT-3 on BASELINE configs[2] shapes: 300 frames x 22 slices of 180x164 px, 256x256 transforms",
                   "l2_policy": "inputs (%.2f GB) and the transform scratch (3.2 GB) larger than L2, no flush" % (d.numel() * 8 / 1e9), "plan": info},
        "kernels_ms": {"all_six_kernels": k_ms},
        "roofline": {"bound": "hbm", "achieved": bytes_min / (k_ms * 1e-3) / 1e9, "peak": peak_hbm, "unit": "GB/s",
                     "frac": bytes_min / (k_ms * 1e-3) / 1e9 / peak_hbm, "traffic": None,
                     "kernel": "motion_stats / fwd_z / lat / peak kernels (whole call)", "kernel_ms": k_ms,
                     "algorithmic_bytes": bytes_min, "bytes_moved_by_design": bytes_moved,
                     "frac_on_bytes_moved": bytes_moved / (k_ms * 1e-3) / 1e9 / peak_hbm, "fft_flop": fft_flop,
                     "fft_tflops": fft_flop / (k_ms * 1e-3) / 1e12, "peak_source": hbm_src},
        "cpu_baseline": cpu, "clocks": clocks,
        "e2e": {"value": n_frames / (e2e_ms * 1e-3), "unit": "frames/s", "h2d_bytes_per_step": int(d.numel() * 8),
                "d2h_bytes_per_step": int(n_frames * 16), "ms_per_step": e2e_ms, "steps": 2},
        "gpu_launches": int(info["launches_last_call"]) * args.steps}))


def run_localize(args):
    """NEXT-4: separable sub-pixel 2-D NCC localization on the projected planes of a
    300-frame ensemble of config 2's shape: 23 + 23 planes of 180 x 164 px per frame (3.26 GB of planes, resident in HBM);
    one step = ulm_rca_localize over the whole ensemble."""
    import torch
    from paper_2511_21647_b200 import Plan, build, fp32_peak_tflops
    torch.cuda.set_device(0)
    build.build()
    cfg = synth.config(2).with_(compound=0)
    kw = rounded_kwargs(cfg)
    n_frames, sig = cfg.n_frames, (1.8, 1.4)
    distinct = synth.bubble_planes(3, 23, 180, 23, 180, 164, seed=6, bubbles_per_plane=5, sigma=sig)
    idx = torch.arange(n_frames, device="cuda") % 3
    d = torch.from_numpy(distinct).cuda()[idx].contiguous()
    warmup = max(args.warmup, 3)
    with Plan(**kw, stage2_block=8, max_frames=n_frames) as plan:
        for _ in range(warmup):
            loc, count = plan.localize(d, sig[0], sig[1], 0.2, 0.7, 16)
        torch.cuda.synchronize()
        sampler = ClockSampler(0)
        sampler.start()
        stream = torch.cuda.current_stream()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        for _ in range(args.steps):
            loc, count = plan.localize(d, sig[0], sig[1], 0.2, 0.7, 16)
        ev1.record(stream)
        torch.cuda.synchronize()
        clocks = sampler.result()
        ms = ev0.elapsed_time(ev1) / args.steps            # includes the allocation / clearing of the result tensors
        info = plan.info()
        h_in = torch.empty(d.shape, dtype=torch.complex64, pin_memory=True)
        h_in.copy_(d)
        d_in = torch.empty_like(d)
        t0 = time.perf_counter()
        for _ in range(2):
            d_in.copy_(h_in, non_blocking=True)
            l2, c2 = plan.localize(d_in, sig[0], sig[1], 0.2, 0.7, 16)
            l_host, c_host = l2.cpu(), c2.cpu()
        e2e_ms = (time.perf_counter() - t0) * 1e3 / 2
        loc, count = loc.cpu().numpy(), count.cpu().numpy()
    byts = float(d.numel() * 8 * 2)                        # planes read twice: frame maximum, then the NCC kernel
    peak_hbm, hbm_src = hbm_peak()
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import localize
        t0 = time.perf_counter()
        ref = localize.localize_frame(distinct[0].astype(np.complex128), 23, 180, 23, 180, 164, sig[0], sig[1], 0.2, 0.7)
        dt = time.perf_counter() - t0
        ok = all(count[0, pl] == len(r) for pl, r in enumerate(ref))
        cpu = {"value": 1 / dt, "unit": "frames/s", "cores": 1, "kind": "oracle",
               "sample": "1 frame = 46 planes (oracle/localize.py, numpy fp64), %.1f s" % dt, "counts_agree": bool(ok)}
    print(json.dumps({
        "metric": "localized frames/s (300-frame ensemble, 46 projected planes per frame)", "value": n_frames / (ms * 1e-3), "unit": "frames/s",
        "n_gpus": 1, "steps": args.steps, "warmup": warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic: synth.bubble_planes, 3 distinct frames tiled over 300 frames",
        "config": {"workload": "SURVEY 8(f) NEXT-4 on BASELINE configs[2] shapes: 300 frames x 46 planes of 180x164 px, 11-tap separable NCC",
                   "l2_policy": "inputs (%.2f GB) larger than L2, no flush" % (d.numel() * 8 / 1e9), "plan": info},
        "localizations_per_frame": float(count.sum()) / n_frames,
        "roofline": {"bound": "hbm", "achieved": byts / (ms * 1e-3) / 1e9, "peak": peak_hbm, "unit": "GB/s",
                     "frac": byts / (ms * 1e-3) / 1e9 / peak_hbm, "traffic": None, "kernel": "localize_max_kernel + localize_kernel (whole call)",
                     "algorithmic_bytes": byts, "peak_source": hbm_src},
        "cpu_baseline": cpu, "clocks": clocks,
        "e2e": {"value": n_frames / (e2e_ms * 1e-3), "unit": "frames/s", "h2d_bytes_per_step": int(d.numel() * 8),
                "d2h_bytes_per_step": int(loc.size * 4 + count.size * 4), "ms_per_step": e2e_ms, "steps": 2},
        "gpu_launches": int(info["launches_last_call"]) * args.steps}))


def run_chain(args):
    """All built steps of the paper's chain on one ensemble, back to back on one stream (context figure, not a BASELINE
    metric): channel data -> per-event slices (Stage 1, compound = 0) -> motion estimation on the slices -> clutter filter
    (in place) -> Stage 2 + compounding + P = 8 sum-projection -> localization.  cfg 2; the paper quotes 0.52 s per
    0.75 s ensemble for its whole pipeline on its GPU, which also contains separation, pairing and tracking."""
    import torch
    from paper_2511_21647_b200 import Plan, build
    torch.cuda.set_device(0)
    build.build()
    cfg = synth.config(2).with_(compound=0)
    n_frames = cfg.n_frames
    channel, host_frames, distinct = make_ensemble(cfg, torch, torch.device("cuda", 0))
    warmup = max(args.warmup, 3)
    with Plan(**rounded_kwargs(cfg), max_frames=n_frames, stage2_block=8, clutter_frames=n_frames, motion_frames=n_frames,
              precision=args.precision) as plan:
        slices = torch.empty((n_frames, plan.slices_complex_per_frame), dtype=torch.complex64, device="cuda")
        planes = torch.empty((n_frames, plan.planes_bytes_per_frame // 8), dtype=torch.complex64, device="cuda")

        def step():
            plan.beamform(channel, out=slices)
            plan.motion_estimate(slices, 0)
            plan.clutter_filter(slices, 4, out=slices)
            plan.stage2_project(slices, out=planes)
            return plan.localize(planes, 1.8, 1.4, 0.2, 0.7, 16)

        for _ in range(warmup):
            step()
        torch.cuda.synchronize()
        sampler = ClockSampler(0)
        sampler.start()
        stream = torch.cuda.current_stream()
        names = ["stage1_per_event", "motion", "clutter", "stage2_projection", "localize"]
        acc = dict.fromkeys(names, 0.0)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        marks = [[torch.cuda.Event(enable_timing=True) for _ in range(6)] for _ in range(args.steps)]
        ev0.record(stream)
        for s in range(args.steps):
            m = marks[s]
            m[0].record(stream); plan.beamform(channel, out=slices)
            m[1].record(stream); plan.motion_estimate(slices, 0)
            m[2].record(stream); plan.clutter_filter(slices, 4, out=slices)
            m[3].record(stream); plan.stage2_project(slices, out=planes)
            m[4].record(stream); plan.localize(planes, 1.8, 1.4, 0.2, 0.7, 16)
            m[5].record(stream)
        ev1.record(stream)
        torch.cuda.synchronize()
        clocks = sampler.result()
        ms = ev0.elapsed_time(ev1) / args.steps
        for m in marks:
            for i, n in enumerate(names):
                acc[n] += m[i].elapsed_time(m[i + 1]) / args.steps
        info = plan.info()
    print(json.dumps({
        "metric": "ensembles through Stage 1 -> motion -> clutter filter -> Stage 2 + projection -> localization (frames/s)",
        "value": n_frames / (ms * 1e-3), "unit": "frames/s", "n_gpus": 1, "steps": args.steps, "warmup": warmup, "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": DTYPE_OF_PRECISION[info["precision"]] + "; later stages f32 (covariance bf16 x 3)",
        "data": "synthetic: cfg 2 channel data (frames %s of the moving scene tiled); no real bubbles or tissue statistics, so the "
                "filter / localizer outputs are not meaningful -- a timing chain only" % (list(distinct),),
        "config": {"workload": "BASELINE configs[2] through every built step of the chain (context; PAPER.md:5 quotes 520 ms per "
                               "ensemble for the paper's whole pipeline on its GPU)", "plan": info},
        "stage_ms": acc, "acquisition_ms": 1e3 * n_frames / cfg.frame_rate_hz, "paper_whole_pipeline_ms": 520.0,
        "clocks": clocks, "gpu_launches": None}))


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
        "scaling": "weak", "vs_baseline": None, "dtype": "f32 (fp32 rows unpacked from the staged IQ entries, fp32 weight)",
        "data": "synthetic: config 1 frame rendered by synth/",
        "config": {"workload": "BASELINE.json configs[4]: 180x180x164 voxels, 11+11 angles, 128+128 RCA, 1 frame"},
        "gather_samples_per_s": gathers / (ms * 1e-3),
        "projection_path_ms_same_frame": ms_proj, "volume_over_projection_time": ms / ms_proj,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": NOMINAL_FP32_TFLOPS, "unit": "TFLOP/s",
                     "frac": achieved / NOMINAL_FP32_TFLOPS, "traffic": capture_traffic("r02_cfg4_volume"),
                     "kernel": "das_volume_mirror_kernel<3,0> (das_volume_kernel<4,0> when the planes / angles are not mirror-symmetric)"},
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


def launch_ranks(args):
    """`--gpus N` without a launcher (WORLD_SIZE unset): start the N ranks through torch.distributed.run -- the
    command the driver uses -- and pass their output and exit code through.  Fails (exit 2) when fewer than N GPUs are
    visible instead of silently running one."""
    import subprocess
    if not args.selftest_launch:
        import torch
        have = torch.cuda.device_count()
        if have < args.gpus:
            sys.stderr.write("bench.py: --gpus %d but only %d CUDA device(s) are visible\n" % (args.gpus, have))
            return 2
    port = 29500 + (os.getpid() * 7) % 2000
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")        # the rank / topology lines show that N ranks really formed
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.run(cmd, env=env).returncode


def run_selftest_launch(args):
    """CPU stand-in for the multi-rank run (tests/test_multirank_cpu.py): the same launch path and rank bookkeeping
    as run_ours -- process group (gloo), barrier, max over ranks, rank 0 prints ONE line -- with a sleep for the
    kernels.  Hidden flag; never a bench value."""
    import torch
    import torch.distributed as dist
    rank, _, world = dist_env()
    if world > 1:
        dist.init_process_group("gloo")
        dist.barrier()
    ms_local = 10.0 * (rank + 1)
    time.sleep(ms_local * 1e-3)

    def all_max(x):
        v = torch.tensor([x], dtype=torch.float64)
        dist.all_reduce(v, op=dist.ReduceOp.MAX)
        return float(v[0])

    fps, ms = whole_job(300, world, ms_local, all_max)
    if world > 1:
        dist.barrier()
    if rank == 0:
        print(json.dumps({"selftest": True, "n_gpus": world, "value": fps, "ms_per_step": ms, "unit": "frames/s"}))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=[2, 3, 4])
    ap.add_argument("--workload", default="beamform", choices=["beamform", "stage2", "clutter", "motion", "localize", "chain"],
                    help="beamform = the BASELINE metric (Stage 1); stage2 = SURVEY 8(f) NEXT-1 on config 2's shapes")
    ap.add_argument("--precision", type=int, default=0, choices=[0, 1, 2, 3],
                    help="scratch format of the main arm (ulm_rca_options.precision; 0 = the library's default)")
    ap.add_argument("--no-arms", action="store_true", help="skip the other scratch formats (roofline_full, ...)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--ref-frames", type=int, default=1)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--per-angle", action="store_true",
                    help="compound = 0: one slice per transmit event (the paper's S_k) instead of the compounded "
                         "projections -- a secondary figure, not the BASELINE metric")
    ap.add_argument("--selftest-launch", action="store_true", help=argparse.SUPPRESS)
    args = ap.parse_args()
    if args.steps < 1 or args.gpus < 1:
        ap.error("--steps and --gpus must be >= 1")
    _, _, world = dist_env()
    if "WORLD_SIZE" not in os.environ and args.gpus > 1 and not (args.impl == "reference"):
        sys.exit(launch_ranks(args))
    if world != args.gpus and args.impl != "reference":
        sys.stderr.write("bench.py: --gpus %d but the launcher started %d rank(s)\n" % (args.gpus, world))
        sys.exit(2)
    if args.selftest_launch:
        run_selftest_launch(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.workload == "stage2":
        run_stage2(args)
    elif args.workload == "clutter":
        run_clutter(args)
    elif args.workload == "motion":
        run_motion(args)
    elif args.workload == "localize":
        run_localize(args)
    elif args.workload == "chain":
        run_chain(args)
    elif args.config == 4:
        run_volume(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- throughput of the Shack-Hartmann WFS hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]

One "step" = one pass of the whole hot path (H1..H8, include/shwfs.h) over one batch of synthetic
input of the headline workload, config 4 of BASELINE.json: 6 LGS WFS x 4632 valid subapertures
(80x80 grid, 10x10 px, pad 32, elongation, 2x2 binning, tau = 0.1) x 100 frames = 2 779 200 spots.
`value` is subaperture-spots/s with inputs resident in HBM; `e2e` is the same through
shwfs_measure_host from pinned host buffers (H2D of every frame and D2H of the slopes inside the timed
region).  Prints ONE JSON line on rank 0.  DESIGN.md section 8 explains every field.

`--impl reference` times the float64 CPU oracle (oracle/, as it stands) on a bounded sample of the
same workload -- the only other place this file runs anything under oracle/ is the `cpu_baseline` leg.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import numpy as np

# ---- constants of the roofline ----------------------------------------------
# algorithmic flops per spot: F_alg (pruned first FFT + frame-paired convolution FFTs)
# and F_nom (1 or 3 full complex P x P FFTs at 5 L log2 L per length-L line)
F_ALG = {1: 7680, 2: 38400, 3: 84800, 4: 84800, 5: 399360}
F_NOM = {1: 10240, 2: 51200, 3: 153600, 4: 153600, 5: 737280}
# FP32 CUDA-core peak derived from unit counts and clocks (B200_PROFILING.md: 148 SMs, 1965 MHz; 128 FP32
# lanes per SM, FMA = 2 flop): 148 * 128 * 2 * 1.965e9.  Measured FFMA chain on this pool: 72.4 TFLOP/s
# (profiles/r01_fp32_peak.md).
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
# sm__pipe_fma_cycles_active (fraction of peak) of the dominant kernel in the committed ncu --set full captures
NCU_FMA_PIPE_ACTIVE = {2: 0.472, 3: 0.636, 4: 0.636, 5: 0.618}
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
# `ncu --set full` captures (profiles/r01_wk10_full_v5.md, r01_wkf16_full.md, r01_pf32_full.md), keyed by config; None where no
# capture of that config's kernel exists.
NCU_TRAFFIC_BYTES_PER_LAUNCH = {2: 129117696 + 4491776, 3: 206465280 + 5998336, 4: 206465280 + 5998336,
                                5: 506622720 + 6679808}


def _dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


class ClockSampler:
    """Polls SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.01):
        self.samples, self.reasons, self.period, self._stop = [], set(), period_s, threading.Event()
        self.max_mhz, self.ok = None, False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # NVML missing: report that instead of inventing clocks
            self.err = repr(e)
        self.th = threading.Thread(target=self._run, daemon=True)

    _NAMES = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
              0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
              0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
                    else int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in self._NAMES.items():
                    if r & bit and name != "gpu_idle":
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self.ok:
            self.th.start()

    def stop(self):
        self._stop.set()
        if self.ok:
            self.th.join(timeout=2)
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "note": "no NVML samples"}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def f_alg(c, L):
    """Algorithmic flops per spot.  Single layer: SURVEY.md 8(d).  With L sodium sub-layers (8(f) f1) the
    cheapest formulation of the same result is L input-pruned first transforms (5 P log2 P (n + P) each), the
    intensities piled up, then ONE frame-paired convolution FFT pair (10 P^2 log2 P per spot)."""
    if L <= 0:
        return F_ALG[c.cfg]
    lg = int(np.log2(c.P))
    return L * 5 * c.P * lg * (c.n + c.P) + (10 * c.P * c.P * lg if c.elong_max_arcsec > 0 else 0)


def workload_name(c, L=0, flux=0.0):
    el = f", elongation <= {c.elong_max_arcsec:g} arcsec" if c.elong_max_arcsec > 0 else ""
    if L > 0:
        el = f", {L} sodium sub-layers (own wavefront each) + round {c.fwhm_short_arcsec:g} arcsec spot kernel"
    if flux > 0:
        el += ", photon + read noise"
    return (f"config{c.cfg} ({c.name}): {c.W} WFS x {c.S}x{c.S} subapertures of {c.n}x{c.n} px on a {c.N}x{c.N} pupil, "
            f"pad {c.P}, {c.b}x{c.b} binning, tau={c.tau:g}{el}, {c.batch}-frame batches")


# ---------------------------------------------------------------------------------------------------
def run_reference(args):
    """The oracle as it stands on the host cores, K steps of a bounded sample (rank 0 only)."""
    rank, _, world = _dist_env()
    if rank != 0:
        return
    from oracle import shwfs_oracle as O
    from paper_1408_0698_b200 import workloads as W
    c = W.CONFIGS[args.config]
    amp = W.pupil_mask(c)
    yx = O.valid_list(amp, c.n, c.min_illum)
    K = W.elongation_kernels(c, 0, yx)
    frames = args.ref_frames
    ph = W.phase_frames(c, 0, range(frames))
    cores = O.max_threads()
    for _ in range(max(args.warmup, 1)):
        O.measure(ph[:1], amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        O.measure(ph, amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K)
    dt = time.perf_counter() - t0
    spots = frames * len(yx)
    v = spots * args.steps / dt
    sample = f"WFS 0, {frames} frame(s) x {len(yx)} valid subapertures = {spots} spots per step"
    print(json.dumps({
        "impl": "reference", "metric": "subaperture_spots_per_s", "value": v, "unit": "spots/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(c), "sample": sample},
        "cpu_baseline": {"value": v, "unit": "spots/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "spots/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ---------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1408_0698_b200 import binding as B, workloads as W
    from paper_1408_0698_b200.distributed import job_throughput, max_over_ranks, rank_frames

    rank, local_rank, world = _dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    c = W.CONFIGS[args.config]
    frames = c.batch
    # one handle per WFS (elongation kernels differ by launch point, reading A13), synthetic frames in HBM
    L = args.sublayers
    my_frames = rank_frames(c.T, frames, rank, world)          # each rank owns its own batch of the stream
    if L > 0:
        # the paper's full LGS model ("MAORY configuration and 3 sodium sub-layers"): every
        # sub-layer has its own wavefront, the elongation comes from the geometry, the kernel is the spot size
        with B.from_config(c, 0, kernels=None) as probe:
            yx = probe.valid_yx
        Ksp = W.spot_size_kernels(c, yx, device=dev)
        sensors = [B.from_config(c, w, kernels=Ksp, valid_yx=yx) for w in range(c.W)]
        for w, s in enumerate(sensors):
            sod = W.sodium_layers(c, w, L)
            s.set_sodium(sod["weight"], sod["defocus"], sod["tilt_x"], sod["tilt_y"], (sod["cx"], sod["cy"]))
        del Ksp
        layer_frames = [int(t) * L + l for t in my_frames for l in range(L)]
        phase = [W.phase_frames_device(c, w, layer_frames, dev).view(frames, L, c.N, c.N) for w in range(c.W)]
    else:
        sensors = [B.from_config(c, w) for w in range(c.W)]
        phase = [W.phase_frames_device(c, w, my_frames, dev) for w in range(c.W)]
    if args.noise_flux > 0:
        for w, s in enumerate(sensors):
            s.set_noise(args.noise_flux / c.n ** 2, args.read_noise, 14080698 + w)
    nsub = sensors[0].nsub
    slopes = [torch.empty((frames, nsub, 2), dtype=torch.float32, device=dev) for _ in range(c.W)]
    spots_per_step = c.W * frames * nsub
    in_bytes = sum(p.numel() * 4 for p in phase)
    out_bytes = sum(s.numel() * 4 for s in slopes)
    stream = torch.cuda.Stream(dev)

    # closed-loop neighbours: DM of --dm-modes modes, residual fused into the gather
    Mdm = args.dm_modes
    if Mdm > 0:
        modes = W.dm_modes_device(c, Mdm, dev)
        for s in sensors:
            s.set_dm(modes)
        del modes
        gen = torch.Generator(device=dev); gen.manual_seed(1408)
        coef = [torch.randn((frames, Mdm), device=dev, generator=gen) * 0.2 for _ in range(c.W)]
        Rmat = [torch.randn((Mdm, 2 * nsub), device=dev, generator=gen) / nsub for _ in range(c.W)]
        cstate = [torch.zeros(Mdm, device=dev) for _ in range(c.W)]

    def step(events=None):
        for w, s in enumerate(sensors):
            if events is not None:
                e0 = torch.cuda.Event(enable_timing=True); e0.record(stream)
            if Mdm > 0 and args.closed_loop:
                with torch.cuda.stream(stream):
                    s.closed_loop(phase[w], Rmat[w], 0.3, cstate[w], want_history=False, stream=stream)
            elif Mdm > 0:
                s.measure_residual(phase[w], coef[w], out=slopes[w], stream=stream)
            else:
                s.measure(phase[w], out=slopes[w], stream=stream)
            if events is not None:
                e1 = torch.cuda.Event(enable_timing=True); e1.record(stream)
                events.append((e0, e1))

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- device-resident throughput
    with torch.cuda.stream(stream):
        for _ in range(max(args.warmup, 3)):
            step()
    barrier()
    sampler = ClockSampler(local_rank)
    l0 = sum(s.launch_count for s in sensors)
    ev = []
    t_beg, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.start()
    with torch.cuda.stream(stream):
        t_beg.record(stream)
        for _ in range(args.steps):
            step(ev)
        t_end.record(stream)
    barrier()
    clocks = sampler.stop()
    launches = sum(s.launch_count for s in sensors) - l0
    ms_total = t_beg.elapsed_time(t_end)
    kern_ms = float(np.mean([a.elapsed_time(b) for a, b in ev]))
    ms_total = max_over_ranks(ms_total, dev)
    value = job_throughput(spots_per_step, args.steps, ms_total, world)

    if Mdm > 0:
        # no host-buffer entry point for the loop calls: report the device-resident numbers only
        if rank == 0:
            spots_per_launch = frames * nsub
            print(json.dumps({
                "metric": "subaperture_spots_per_s", "value": value, "unit": "spots/s", "n_gpus": world,
                "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_total / args.steps,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": workload_name(c, L, args.noise_flux) + f", DM of {Mdm} modes, " +
                           ("sequential pure-integrator loop (shwfs_closed_loop)" if args.closed_loop
                            else "residual fused into the gather (shwfs_measure_residual)"),
                           "spots_per_step_per_gpu": spots_per_step},
                "wfs_frames_per_s": value / nsub, "loop_steps_per_s_per_wfs": value / nsub if args.closed_loop else None,
                "ms_per_wfs_call": kern_ms, "clocks": clocks, "e2e": None, "gpu_launches": int(launches),
                "dm_flops_per_spot": 2 * Mdm * c.n * c.n,
                "dm_tflops": 2 * Mdm * c.n * c.n * spots_per_launch / (kern_ms * 1e-3) / 1e12}))
        for s in sensors:
            s.close()
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- end to end from pinned host memory through shwfs_measure_host
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    h_phase = [torch.empty(tuple(phase[0].shape), dtype=torch.float32, pin_memory=True) for _ in range(c.W)]
    for w in range(c.W):
        h_phase[w].copy_(phase[w])
    h_slopes = [torch.empty((frames, nsub, 2), dtype=torch.float32, pin_memory=True) for _ in range(c.W)]
    for w, s in enumerate(sensors):                       # warm-up: allocates the staging buffers
        s.measure_host(h_phase[w], out=h_slopes[w])
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        for w, s in enumerate(sensors):                   # the W sensors of the system back to back on the bus
            s.measure_host_async(h_phase[w], h_slopes[w])
        for s in sensors:
            s.host_wait()
    torch.cuda.synchronize(dev)
    e2e_s = time.perf_counter() - t0
    e2e_value = job_throughput(spots_per_step, e2e_steps, 1e3 * max_over_ranks(e2e_s, dev), world)
    e2e_check = float((h_slopes[0].to(dev) - slopes[0]).abs().max().item())

    if rank == 0:
        spots_per_launch = frames * nsub
        fa = f_alg(c, L)
        ach = fa * spots_per_launch / (kern_ms * 1e-3) / 1e12
        roofline = {"bound": "alu", "achieved": ach, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                    "frac": ach / FP32_PEAK_TFLOPS, "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH.get(c.cfg) if L <= 0 and args.noise_flux <= 0 else None,
                    "kernel": {B.ALGO_WK: f"wk_measure_kernel<{c.n}>", B.ALGO_WK_FFT: f"wkf_kernel<{c.n}>", B.ALGO_PRUNED_FFT: f"pruned_fft_kernel<{c.P}>",
                               B.ALGO_LITERAL: f"literal_kernel<{c.P}>"}.get(sensors[0].algorithm, f"algo{sensors[0].algorithm}"),
                    "kernel_ms": kern_ms, "spots_per_launch": spots_per_launch,
                    "flops_per_spot": fa, "flops_basis": "F_alg (SURVEY.md 8(d))" if L <= 0 else
                    "L pruned first FFTs + one frame-paired convolution pair (DESIGN.md 7)",
                    "frac_nominal_fft_flops": (F_NOM[c.cfg] * spots_per_launch / (kern_ms * 1e-3) / 1e12 / FP32_PEAK_TFLOPS
                                               if L <= 0 else None),
                    "peak_basis": "derived: 148 SM x 128 lanes x 2 x 1.965 GHz (measured FFMA chain 72.4)",
                    "fma_pipe_active_ncu": NCU_FMA_PIPE_ACTIVE.get(c.cfg) if L <= 0 and args.noise_flux <= 0 else None,
                    "hbm_frac": (in_bytes + out_bytes) / c.W / (kern_ms * 1e-3) / 1e9 / _hbm_peak()}
        cpu = None if args.no_cpu_baseline else cpu_baseline(c, args, phase, sensors[0].valid_yx)
        out = {
            "metric": "subaperture_spots_per_s", "value": value, "unit": "spots/s", "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(c, L, args.noise_flux), "spots_per_step_per_gpu": spots_per_step,
                       "l2": f"inputs larger than L2 ({in_bytes / 1e6:.0f} MB read per step), no flush"},
            "wfs_frames_per_s": value / nsub, "system_frames_per_s": value / nsub / c.W,
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": "spots/s",
                    "h2d_bytes_per_step": sum(s.host_bytes_per_frame * (p.numel() // (c.N * c.N)) for s, p in zip(sensors, phase)),
                    "h2d_note": "only the column runs of valid subapertures cross the bus (shwfs_host_bytes_per_frame); "
                                f"the pinned host tensors hold {in_bytes} bytes",
                    "d2h_bytes_per_step": out_bytes,
                    "steps": e2e_steps, "api": "shwfs_measure_host_async + shwfs_host_wait (one call per WFS)", "max_abs_diff_vs_device_path": e2e_check},
            "gpu_launches": int(launches),
            "roofline": roofline,
            "cpu_baseline": cpu,
        }
        print(json.dumps(out))
    for s in sensors:
        s.close()
    if world > 1:
        dist.destroy_process_group()


def run_pyramid(args):
    """Pyramid WFS: frames/s of pyrwfs_measure on a synthetic LBT-like workload, inputs
    resident in HBM, CUDA events on the launching stream; the numpy oracle on the host cores beside it."""
    import torch
    from paper_1408_0698_b200 import binding as B, workloads as W
    rank, local_rank, world = _dist_env()
    if rank != 0:
        return
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    p = W.PYRAMIDS[args.pyramid]
    amp = W.pyramid_mask(p)
    T = args.pyramid_frames
    ph_host = W.pyramid_frames(p, range(min(T, 8)), 0.3)
    ph = torch.from_numpy(ph_host).to(dev).repeat((T + ph_host.shape[0] - 1) // ph_host.shape[0], 1, 1)[:T].contiguous()
    stream = torch.cuda.Stream(dev)
    with B.Pyrwfs(amp, p.Np, p.s, p.bp, p.r_mod, p.K, p.D_pix) as s:
        out = torch.empty((T, s.nvalid, 2), dtype=torch.float32, device=dev)
        for _ in range(max(args.warmup, 3)):
            s.measure(ph, out=out, stream=stream)
        torch.cuda.synchronize(dev)
        sampler = ClockSampler(local_rank)
        l0 = s.launch_count
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler.start()
        e0.record(stream)
        for _ in range(args.steps):
            s.measure(ph, out=out, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize(dev)
        clocks = sampler.stop()
        ms = e0.elapsed_time(e1)
        launches = s.launch_count - l0
        nvalid = s.nvalid
    value = T * args.steps / (ms * 1e-3)
    Kp = max(p.K, 1)
    lg = int(np.log2(p.Np))
    # nominal flops per frame: per modulation point N pruned row lines, Np columns x 2 transforms, 2N output rows
    lines = Kp * (p.N + 2 * p.Np + 2 * p.N)
    flops = lines * 5 * p.Np * lg
    ach = flops * value / 1e12
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import pyramid as OP
        yx = OP.valid_pixels(amp, p.bp)
        nfr = max(1, min(args.cpu_frames, 4))
        t0 = time.perf_counter()
        OP.measure(ph_host[:nfr], amp, yx, p.Np, p.s, p.bp, p.r_mod, p.K, p.D_pix)
        dt = time.perf_counter() - t0
        cpu = {"value": nfr / dt, "unit": "frames/s", "cores": 1, "kind": "oracle",
               "sample": f"{nfr} frame(s), numpy fft2 oracle, {dt:.1f} s"}
    print(json.dumps({
        "metric": "pyramid_wfs_frames_per_s", "value": value, "unit": "frames/s", "n_gpus": 1, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"pyramid '{p.name}': pupil {p.N} px, pad {p.Np}, separation {p.s}, {p.bp}x{p.bp} binning "
                               f"to {p.N // p.bp}x{p.N // p.bp}, modulation {p.r_mod:g} lambda/D in {p.K} points, "
                               f"{nvalid} valid pixels, {T}-frame batches"},
        "clocks": clocks, "e2e": None, "gpu_launches": int(launches),
        "roofline": {"bound": "alu", "achieved": ach, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                     "frac": ach / FP32_PEAK_TFLOPS, "traffic": None, "kernel": "pyr_cols_kernel (+ rows, final)",
                     "flops_per_frame": flops, "flops_basis": "5 L log2 L per line of the pruned passes (DESIGN.md 14)"},
        "cpu_baseline": cpu}))


def _hbm_peak():
    try:
        return float(json.loads((ROOT / "MEASURED_PEAKS.json").read_text())["hbm_gbs"])
    except Exception:
        return 6650.0   # B200_PROFILING.md fallback


def cpu_baseline(c, args, phase_dev, yx_lib=None):
    """The oracle as it stands on this box's host cores over a bounded sample of the same batch."""
    from oracle import shwfs_oracle as O
    from paper_1408_0698_b200 import workloads as W
    amp = W.pupil_mask(c)
    yx = O.valid_list(amp, c.n, c.min_illum)
    L = args.sublayers
    if L > 0 or args.noise_flux > 0:
        K = W.spot_size_kernels(c, yx) if L > 0 else W.elongation_kernels(c, 0, yx)
        sod = W.sodium_layers(c, 0, max(L, 1))
        kw = dict(weight=sod["weight"] if L > 0 else [1.0], defocus=sod["defocus"] if L > 0 else [0.0],
                  tilt_x=sod["tilt_x"] if L > 0 else None, tilt_y=sod["tilt_y"] if L > 0 else None,
                  cx=sod["cx"], cy=sod["cy"], tau=c.tau, kernels=K,
                  flux=args.noise_flux / c.n ** 2, ron=args.read_noise, seed=14080698)
        run = lambda p: O.measure_lgs(p, amp, yx, c.n, c.P, c.b, c.dx, **kw)
        nfr = max(1, args.cpu_frames // max(L, 1))
    else:
        K = W.elongation_kernels(c, 0, yx)
        run = lambda p: O.measure(p, amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K)
        nfr = args.cpu_frames
    ph = phase_dev[0][:nfr].cpu().numpy()
    run(ph[:1])                                                               # page in / build
    t0 = time.perf_counter()
    run(ph)
    dt = time.perf_counter() - t0
    spots = ph.shape[0] * len(yx)
    return {"value": spots / dt, "unit": "spots/s", "cores": O.max_threads(), "kind": "oracle",
            "sample": f"WFS 0, first {ph.shape[0]} frames of the timed batch = {spots} spots, {dt:.1f} s"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--cpu-frames", type=int, default=100)
    ap.add_argument("--ref-frames", type=int, default=4)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sublayers", type=int, default=0,
                    help="L > 0: the paper's full LGS model, L sodium sub-layers with their own wavefronts (8(f) f1)")
    ap.add_argument("--noise-flux", type=float, default=0.0,
                    help="> 0: detector noise, photo-electrons per fully lit subaperture per frame (8(f) f2)")
    ap.add_argument("--read-noise", type=float, default=3.0)
    ap.add_argument("--dm-modes", type=int, default=0,
                    help="M > 0: subtract a DM of M modes inside the gather (8(f) f3, shwfs_measure_residual)")
    ap.add_argument("--pyramid", default=None, choices=["tiny", "lbt"],
                    help="time the pyramid WFS (8(f) f4) on this workloads.PYRAMIDS entry instead of the SH path")
    ap.add_argument("--pyramid-frames", type=int, default=32)
    ap.add_argument("--closed-loop", action="store_true",
                    help="with --dm-modes: run the batch as sequential pure-integrator frames (shwfs_closed_loop)")
    args = ap.parse_args()
    if args.pyramid:
        run_pyramid(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

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
# Figures that only a profiler can give (FMA-pipe activity, DRAM bytes and executed FP32 flops per launch of the
# dominant kernel) live in profiles/ncu_constants.json, keyed by the kernel instance name the library reports
# (shwfs_last_kernel) and stamped with a hash of the sources they were captured at.  They are printed as
# "not measured in this run" values and become null the moment the sources change (profiles/ncu_constants.md).
NCU_JSON = ROOT / "profiles" / "ncu_constants.json"


def sources_sha1(paths):
    """sha1 over the CODE of the named source files (relative to the repo root), in the order given: C comments
    and white space are dropped first, so that rewording a comment does not disown a capture but any change a
    compiler could see does."""
    import hashlib
    import re
    h = hashlib.sha1()
    for rel in paths:
        text = (ROOT / rel).read_text()
        text = re.sub(r"/\*.*?\*/", " ", text, flags=re.S)
        text = re.sub(r"//[^\n]*", " ", text)
        h.update(rel.encode() + b"\0" + "".join(text.split()).encode())
    return h.hexdigest()


def ncu_constants(kernel):
    """The committed ncu figures of `kernel`, or (None, why) if there are none for the sources as they stand."""
    try:
        table = json.loads(NCU_JSON.read_text())["kernels"]
    except Exception as e:
        return None, f"profiles/ncu_constants.json unreadable: {e!r}"
    ent = table.get(kernel)
    if ent is None:
        return None, f"no ncu capture of {kernel} committed"
    try:
        now = sources_sha1(ent["sources"])
    except Exception as e:
        return None, f"sources of the capture unreadable: {e!r}"
    if now != ent["sources_sha1"]:
        return None, f"sources changed since the capture ({ent['capture']}): figures withheld"
    return ent, f"from {ent['capture']} (ncu, not measured in this run)"


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
class Workload:
    """One config of BASELINE.json on this rank: handles (one per WFS), synthetic frames resident in HBM, outputs."""

    def __init__(self, c, args, L, dev, rank=0, world=1, dm_modes=0, noise_flux=0.0):
        import torch
        from paper_1408_0698_b200 import binding as B, workloads as W
        from paper_1408_0698_b200.distributed import rank_frames
        self.c, self.L, self.dev, self.torch = c, L, dev, torch
        frames = self.frames = c.batch
        my_frames = rank_frames(c.T, frames, rank, world)          # each rank owns its own batch of the stream
        if L > 0:
            # the paper's full LGS model ("MAORY configuration and 3 sodium sub-layers"): every
            # sub-layer has its own wavefront, the elongation comes from the geometry, the kernel is the spot size
            with B.from_config(c, 0, kernels=None) as probe:
                yx = probe.valid_yx
            Ksp = W.spot_size_kernels(c, yx, device=dev)
            self.sensors = [B.from_config(c, w, kernels=Ksp, valid_yx=yx) for w in range(c.W)]
            for w, s in enumerate(self.sensors):
                sod = W.sodium_layers(c, w, L)
                s.set_sodium(sod["weight"], sod["defocus"], sod["tilt_x"], sod["tilt_y"], (sod["cx"], sod["cy"]))
            del Ksp
            layer_frames = [int(t) * L + l for t in my_frames for l in range(L)]
            self.phase = [W.phase_frames_device(c, w, layer_frames, dev).view(frames, L, c.N, c.N) for w in range(c.W)]
        else:
            self.sensors = [B.from_config(c, w) for w in range(c.W)]
            self.phase = [W.phase_frames_device(c, w, my_frames, dev) for w in range(c.W)]
        if noise_flux > 0:
            for w, s in enumerate(self.sensors):
                s.set_noise(noise_flux / c.n ** 2, args.read_noise, 14080698 + w, photon_model=args.photon_model)
        self.nsub = self.sensors[0].nsub
        self.slopes = [torch.empty((frames, self.nsub, 2), dtype=torch.float32, device=dev) for _ in range(c.W)]
        self.spots_per_step = c.W * frames * self.nsub
        self.in_bytes = sum(p.numel() * 4 for p in self.phase)
        self.out_bytes = sum(s.numel() * 4 for s in self.slopes)
        self.stream = torch.cuda.Stream(dev)
        # closed-loop neighbours: DM of dm_modes modes, residual fused into the gather
        self.Mdm = dm_modes
        if dm_modes > 0:
            modes = W.dm_modes_device(c, dm_modes, dev)
            for s in self.sensors:
                s.set_dm(modes)
            del modes
            gen = torch.Generator(device=dev); gen.manual_seed(1408)
            self.coef = [torch.randn((frames, dm_modes), device=dev, generator=gen) * 0.2 for _ in range(c.W)]
            self.Rmat = [torch.randn((dm_modes, 2 * self.nsub), device=dev, generator=gen) / self.nsub for _ in range(c.W)]
            self.cstate = [torch.zeros(dm_modes, device=dev) for _ in range(c.W)]

    def step(self, events=None, closed_loop=False):
        torch, stream = self.torch, self.stream
        for w, s in enumerate(self.sensors):
            if events is not None:
                e0 = torch.cuda.Event(enable_timing=True); e0.record(stream)
            if self.Mdm > 0 and closed_loop:
                with torch.cuda.stream(stream):
                    s.closed_loop(self.phase[w], self.Rmat[w], 0.3, self.cstate[w], want_history=False, stream=stream)
            elif self.Mdm > 0:
                s.measure_residual(self.phase[w], self.coef[w], out=self.slopes[w], stream=stream)
            else:
                s.measure(self.phase[w], out=self.slopes[w], stream=stream)
            if events is not None:
                e1 = torch.cuda.Event(enable_timing=True); e1.record(stream)
                events.append((e0, e1))

    def time_device(self, steps, warmup, barrier, sampler=None, closed_loop=False):
        """W warm-up steps, then K timed steps bracketed by barrier + synchronize on both sides.  Returns total ms
        (CUDA events on the launching stream), mean ms of one handle's call, kernels launched."""
        torch, stream = self.torch, self.stream
        with torch.cuda.stream(stream):
            for _ in range(warmup):
                self.step(closed_loop=closed_loop)
        barrier()
        l0 = sum(s.launch_count for s in self.sensors)
        ev = []
        t_beg, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        if sampler is not None:
            sampler.start()
        with torch.cuda.stream(stream):
            t_beg.record(stream)
            for _ in range(steps):
                self.step(ev, closed_loop=closed_loop)
            t_end.record(stream)
        barrier()
        clocks = sampler.stop() if sampler is not None else None
        launches = sum(s.launch_count for s in self.sensors) - l0
        return t_beg.elapsed_time(t_end), float(np.mean([a.elapsed_time(b) for a, b in ev])), int(launches), clocks

    def time_e2e(self, steps, barrier):
        """The same measurement through shwfs_measure_host_async + shwfs_host_wait from pinned host tensors: H2D of
        every frame and D2H of the slopes inside the timed region.  Returns seconds, max |host path - device path|."""
        torch, c = self.torch, self.c
        h_phase = [torch.empty(tuple(self.phase[0].shape), dtype=torch.float32, pin_memory=True) for _ in range(c.W)]
        for w in range(c.W):
            h_phase[w].copy_(self.phase[w])
        h_slopes = [torch.empty((self.frames, self.nsub, 2), dtype=torch.float32, pin_memory=True) for _ in range(c.W)]
        for w, s in enumerate(self.sensors):                  # warm-up: allocates the staging buffers
            s.measure_host(h_phase[w], out=h_slopes[w])
        barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            for w, s in enumerate(self.sensors):              # the W sensors of the system back to back on the bus
                s.measure_host_async(h_phase[w], h_slopes[w])
            for s in self.sensors:
                s.host_wait()
        torch.cuda.synchronize(self.dev)
        dt = time.perf_counter() - t0
        check = float((h_slopes[0].to(self.dev) - self.slopes[0]).abs().max().item())
        return dt, check

    def h2d_bytes_per_step(self):
        c = self.c
        return sum(s.host_bytes_per_frame * (p.numel() // (c.N * c.N)) for s, p in zip(self.sensors, self.phase))

    def roofline(self, kern_ms):
        """F_alg x spots per launch / mean launch duration against the derived FP32 peak; beside
        it the kernel's own executed FP32 flops (from the committed ncu capture of that kernel instance)."""
        c, L = self.c, self.L
        spots_per_launch = self.frames * self.nsub
        fa = f_alg(c, L)
        ach = fa * spots_per_launch / (kern_ms * 1e-3) / 1e12
        kernel = self.sensors[0].last_kernel
        ent, note = ncu_constants(kernel)
        fx = ent.get("fp32_flops_per_spot") if ent else None
        return {"bound": "alu", "achieved": ach, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                "frac": ach / FP32_PEAK_TFLOPS,
                "traffic": ent.get("dram_bytes_per_launch") if ent else None,
                "kernel": kernel, "kernel_ms": kern_ms, "spots_per_launch": spots_per_launch,
                "flops_per_spot": fa, "flops_basis": "F_alg (SURVEY.md 8(d))" if L <= 0 else
                "L pruned first FFTs + one frame-paired convolution pair (DESIGN.md 7)",
                "frac_nominal_fft_flops": (F_NOM[c.cfg] * spots_per_launch / (kern_ms * 1e-3) / 1e12 / FP32_PEAK_TFLOPS
                                           if L <= 0 else None),
                "frac_executed": (fx * spots_per_launch / (kern_ms * 1e-3) / 1e12 / FP32_PEAK_TFLOPS) if fx else None,
                "flops_executed_per_spot_ncu": fx,
                "peak_basis": "derived: 148 SM x 128 lanes x 2 x 1.965 GHz (measured FFMA chain 72.4)",
                "fma_pipe_active_ncu": ent.get("fma_pipe_active") if ent else None,
                "ncu_note": note,
                "hbm_frac": (self.in_bytes + self.out_bytes) / c.W / (kern_ms * 1e-3) / 1e9 / _hbm_peak()}

    def close(self):
        for s in self.sensors:
            s.close()
        self.phase = self.slopes = None
        self.torch.cuda.empty_cache()


def per_config_entry(cfg_id, L, args, dev, barrier, steps):
    """One extra workload of the default run: device-resident throughput and roofline of config `cfg_id` (with L
    sodium sub-layers if L > 0), a few steps, same timing protocol as the headline."""
    from paper_1408_0698_b200 import workloads as W
    c = W.CONFIGS[cfg_id]
    wl = Workload(c, args, L, dev)
    try:
        ms_total, kern_ms, launches, _ = wl.time_device(steps, 3, barrier)
        value = wl.spots_per_step * steps / (ms_total * 1e-3)
        r = wl.roofline(kern_ms)
        return {"workload": workload_name(c, L), "value": value, "unit": "spots/s", "steps": steps, "warmup": 3,
                "wfs_frames_per_s": value / wl.nsub, "system_frames_per_s": value / wl.nsub / c.W,
                "kernel": r["kernel"], "kernel_ms": kern_ms, "gpu_launches": launches,
                "roofline": {k: r[k] for k in ("frac", "frac_executed", "frac_nominal_fft_flops", "flops_per_spot",
                                               "flops_executed_per_spot_ncu", "fma_pipe_active_ncu", "traffic",
                                               "ncu_note")},
                "target_50pct_spots_per_s": 0.5 * FP32_PEAK_TFLOPS * 1e12 / f_alg(c, L)}
    finally:
        wl.close()


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1408_0698_b200 import workloads as W
    from paper_1408_0698_b200.distributed import job_throughput, max_over_ranks

    rank, local_rank, world = _dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    c = W.CONFIGS[args.config]
    L, Mdm = args.sublayers, args.dm_modes
    wl = Workload(c, args, L, dev, rank, world, dm_modes=Mdm, noise_flux=args.noise_flux)
    nsub, frames, spots_per_step = wl.nsub, wl.frames, wl.spots_per_step
    warm = max(args.warmup, 3)

    # ---- device-resident throughput
    ms_total, kern_ms, launches, clocks = wl.time_device(args.steps, warm, barrier, ClockSampler(local_rank),
                                                         closed_loop=args.closed_loop)
    ms_total = max_over_ranks(ms_total, dev)
    value = job_throughput(spots_per_step, args.steps, ms_total, world)

    if Mdm > 0:
        # no host-buffer entry point for the loop calls: report the device-resident numbers only
        if rank == 0:
            spots_per_launch = frames * nsub
            print(json.dumps({
                "metric": "subaperture_spots_per_s", "value": value, "unit": "spots/s", "n_gpus": world,
                "steps": args.steps, "warmup": warm, "ms_per_step": ms_total / args.steps,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": workload_name(c, L, args.noise_flux) + f", DM of {Mdm} modes, " +
                           ("sequential pure-integrator loop (shwfs_closed_loop)" if args.closed_loop
                            else "residual fused into the gather (shwfs_measure_residual)"),
                           "spots_per_step_per_gpu": spots_per_step},
                "wfs_frames_per_s": value / nsub, "loop_steps_per_s_per_wfs": value / nsub if args.closed_loop else None,
                "ms_per_wfs_call": kern_ms, "clocks": clocks, "e2e": None, "gpu_launches": int(launches),
                "dm_flops_per_spot": 2 * Mdm * c.n * c.n,
                "dm_tflops": 2 * Mdm * c.n * c.n * spots_per_launch / (kern_ms * 1e-3) / 1e12}))
        wl.close()
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- end to end from pinned host memory through shwfs_measure_host
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    e2e_s, e2e_check = wl.time_e2e(e2e_steps, barrier)
    e2e_value = job_throughput(spots_per_step, e2e_steps, 1e3 * max_over_ranks(e2e_s, dev), world)

    if rank == 0:
        roofline = wl.roofline(kern_ms)
        cpu = None if args.no_cpu_baseline else cpu_baseline(c, args, wl.phase, wl.sensors[0].valid_yx)
        out = {
            "metric": "subaperture_spots_per_s", "value": value, "unit": "spots/s", "n_gpus": world,
            "steps": args.steps, "warmup": warm, "ms_per_step": ms_total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(c, L, args.noise_flux), "spots_per_step_per_gpu": spots_per_step,
                       "l2": f"inputs larger than L2 ({wl.in_bytes / 1e6:.0f} MB read per step), no flush"},
            "wfs_frames_per_s": value / nsub, "system_frames_per_s": value / nsub / c.W,
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": "spots/s",
                    "h2d_bytes_per_step": wl.h2d_bytes_per_step(),
                    "h2d_note": "only the column runs of valid subapertures cross the bus (shwfs_host_bytes_per_frame); "
                                f"the pinned host tensors hold {wl.in_bytes} bytes",
                    "d2h_bytes_per_step": wl.out_bytes,
                    "steps": e2e_steps, "api": "shwfs_measure_host_async + shwfs_host_wait (one call per WFS)", "max_abs_diff_vs_device_path": e2e_check},
            "gpu_launches": int(launches),
            "roofline": roofline,
            "cpu_baseline": cpu,
        }
    wl.close()
    if rank == 0:
        # ---- the other north_star configs and the paper's own timing case, a few steps each (single GPU, default run)
        if args.per_config and world == 1 and L <= 0 and args.noise_flux <= 0:
            pc = {}
            for key, cfg_id, Lx in (("2", 2, 0), ("3", 3, 0), ("5", 5, 0), ("4_sublayers3", 4, 3)):
                if cfg_id == args.config and Lx == 0:
                    continue
                try:
                    pc[key] = per_config_entry(cfg_id, Lx, args, dev, barrier, args.per_config_steps)
                except Exception as e:     # a failed extra never takes the headline line down with it
                    pc[key] = {"error": repr(e)}
            out["per_config"] = pc
            if not args.no_cpu_baseline:
                out["cpu_baseline_more"] = cpu_baseline_more(args)
        print(json.dumps(out))
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
    pent, pnote = ncu_constants(f"pyr_cols_kernel<{32 if p.Np == 1024 else 16}>")
    print(json.dumps({
        "metric": "pyramid_wfs_frames_per_s", "value": value, "unit": "frames/s", "n_gpus": 1, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"pyramid '{p.name}': pupil {p.N} px, pad {p.Np}, separation {p.s}, {p.bp}x{p.bp} binning "
                               f"to {p.N // p.bp}x{p.N // p.bp}, modulation {p.r_mod:g} lambda/D in {p.K} points, "
                               f"{nvalid} valid pixels, {T}-frame batches"},
        "clocks": clocks, "e2e": None, "gpu_launches": int(launches),
        "roofline": {"bound": "alu", "achieved": ach, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                     "frac": ach / FP32_PEAK_TFLOPS, "traffic": (pent or {}).get("dram_bytes_per_launch"),
                     "traffic_note": "pyr_cols_kernel, one 16-frame chunk per launch; " + pnote,
                     "fma_pipe_active_ncu": (pent or {}).get("fma_pipe_active"),
                     "kernel": "pyr_cols_kernel (+ rows, final)",
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
                  flux=args.noise_flux / c.n ** 2, ron=args.read_noise, seed=14080698,
                  photon_model=args.photon_model)
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


def cpu_baseline_more(args):
    """SURVEY.md 8(d) 'Oracle timing': the oracle as it stands on config 3 frame 0 in full (4632 spots), on all host
    cores and on one thread, and on 4 frames of config 5 (all cores)."""
    from oracle import shwfs_oracle as O
    from paper_1408_0698_b200 import workloads as W
    out = {}
    all_cores = O.max_threads()
    # the one-thread case goes last: the oracle keeps the thread count it was last given
    for key, cfg_id, nfr, threads in (("config3_frame0_all_cores", 3, 1, 0), ("config5_4frames_all_cores", 5, 4, 0),
                                      ("config3_frame0_one_thread", 3, 1, 1)):
        c = W.CONFIGS[cfg_id]
        amp = W.pupil_mask(c)
        yx = O.valid_list(amp, c.n, c.min_illum)
        K = W.elongation_kernels(c, 0, yx)
        ph = W.phase_frames(c, 0, range(nfr))
        t0 = time.perf_counter()
        O.measure(ph, amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K, nthreads=threads)
        dt = time.perf_counter() - t0
        spots = nfr * len(yx)
        out[key] = {"value": spots / dt, "unit": "spots/s", "cores": threads if threads else all_cores,
                    "kind": "oracle", "sample": f"config {cfg_id}, WFS 0, {nfr} frame(s) = {spots} spots, {dt:.1f} s",
                    "frames_per_s": nfr / dt,
                    "extrapolated_s_per_1000_frames_all_wfs": 1000.0 * c.W * dt / nfr}
    return out


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
    ap.add_argument("--photon-model", type=int, default=0, choices=[0, 1],
                    help="with --noise-flux: 0 = Gaussian limit of the photon noise, 1 = Poisson counts (include/shwfs.h)")
    ap.add_argument("--dm-modes", type=int, default=0,
                    help="M > 0: subtract a DM of M modes inside the gather (8(f) f3, shwfs_measure_residual)")
    ap.add_argument("--pyramid", default=None, choices=["tiny", "lbt"],
                    help="time the pyramid WFS (8(f) f4) on this workloads.PYRAMIDS entry instead of the SH path")
    ap.add_argument("--pyramid-frames", type=int, default=32)
    ap.add_argument("--no-per-config", dest="per_config", action="store_false",
                    help="skip the per_config section (configs 2, 3, 5 and config 4 with 3 sodium sub-layers)")
    ap.add_argument("--per-config-steps", type=int, default=10)
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

"""Small calls of every kernel family through the C ABI, for compute-sanitizer (SURVEY.md sections 4 and 5: "ABI"
and "Race detection" rows).  Not a pytest module: run it under the tool,

    compute-sanitizer --tool memcheck  python tests/sanitizer_workloads.py
    compute-sanitizer --tool racecheck python tests/sanitizer_workloads.py
    compute-sanitizer --tool synccheck python tests/sanitizer_workloads.py
    compute-sanitizer --tool initcheck python tests/sanitizer_workloads.py

(profiles/r02_sanitizer.md keeps the summaries).  Inputs are the seeded generators of workloads.py on explicit
subsets of the valid subapertures, small enough for racecheck; SHWFS_FORCE_PERSISTENT=1 makes the library take its
persistent TMA instances on these small calls.  Every result is also checked for finiteness, so a tool that
serialises the kernels still sees a run that did real work.
"""
import os
import sys
from pathlib import Path

os.environ.setdefault("SHWFS_FORCE_PERSISTENT", "1")
sys.path.insert(0, str(Path(__file__).resolve().parent.parent))

import numpy as np
import torch

from paper_1408_0698_b200 import binding as B, workloads as W


def subset(c, every):
    """every `every`-th valid subaperture of config c (A2 rule evaluated by a throw-away handle)"""
    with B.from_config(c, 0, kernels=None) as probe:
        return probe.valid_yx[::every].copy()


def finite(name, t, kernels):
    assert bool(torch.isfinite(t).all()), name
    print(f"ok {name}: {tuple(t.shape)} {kernels}")


def sensor_cases():
    # create / measure / destroy loop on three geometries, every algorithm that has an instance
    for rep in range(2):
        for cfg_id, every, T in ((1, 1, 4), (2, 30, 3), (3, 70, 40), (5, 70, 3)):
            c = W.CONFIGS[cfg_id]
            yx = subset(c, every)
            K = W.elongation_kernels(c, 0, yx)
            ph = torch.from_numpy(W.phase_frames(c, 0, [t % 2 for t in range(T)])).cuda()
            with B.from_config(c, 0, kernels=K, valid_yx=yx) as s:
                names = []
                for a in (B.ALGO_AUTO, B.ALGO_WK, B.ALGO_WK_GENERIC, B.ALGO_WK_FFT, B.ALGO_PRUNED_FFT, B.ALGO_LITERAL):
                    try:
                        s.algorithm = a
                    except B.ShwfsError as e:
                        assert e.code == B.SHWFS_EUNSUPPORTED
                        continue
                    out = s.measure(ph)
                    names.append(s.last_kernel)
                    finite(f"config {cfg_id} algo {a}", out, s.last_kernel)
                img = s.debug_spots(ph, 2)
                finite(f"config {cfg_id} stage 2", img, s.last_kernel)
    # host-buffer entry point, pageable and pinned
    c = W.CONFIGS[1]
    ph = W.phase_frames(c, 0, range(4))
    with B.from_config(c, 0) as s:
        finite("measure_host", torch.from_numpy(s.measure_host(ph)), s.last_kernel)


def lgs_cases():
    # sodium sub-layers (own wavefronts and shared) + detector noise: the EXT instances
    c = W.CONFIGS[3]
    yx = subset(c, 70)
    K = W.spot_size_kernels(c, yx)
    for L, shared, T in ((3, False, 40), (2, True, 3)):
        sod = W.sodium_layers(c, 0, L)
        shape = (T, c.N, c.N) if shared else (T, L, c.N, c.N)
        ph = torch.from_numpy(W.phase_frames(c, 0, range(2))[:1].repeat(int(np.prod(shape[:-2])), 0).reshape(shape)).cuda()
        with B.from_config(c, 0, kernels=K, valid_yx=yx) as s:
            s.set_sodium(sod["weight"], sod["defocus"], sod["tilt_x"], sod["tilt_y"], (sod["cx"], sod["cy"]), shared_phase=shared)
            s.set_noise(5.0, 3.0, 1408)
            for a in (B.ALGO_WK, B.ALGO_WK_GENERIC):
                s.algorithm = a
                finite(f"lgs L={L} shared={shared} algo {a}", s.measure(ph), s.last_kernel)
    c = W.CONFIGS[5]
    yx = subset(c, 70)
    K = W.spot_size_kernels(c, yx)
    sod = W.sodium_layers(c, 0, 3)
    ph = torch.from_numpy(W.phase_frames(c, 0, range(1)).repeat(6, 0).reshape(2, 3, c.N, c.N)).cuda()
    with B.from_config(c, 0, kernels=K, valid_yx=yx) as s:
        s.set_sodium(sod["weight"], sod["defocus"], sod["tilt_x"], sod["tilt_y"], (sod["cx"], sod["cy"]))
        finite("lgs n=16 L=3 (wkf multi-layer)", s.measure(ph), s.last_kernel)


def loop_cases():
    # DM residual: tensor-core GEMM (T > 8), FP32 GEMV (T <= 8), reconstructor, closed loop
    c = W.CONFIGS[3]
    yx = subset(c, 70)
    K = W.elongation_kernels(c, 0, yx)
    M = 16
    modes = torch.from_numpy(W.dm_modes(c, M)).cuda()
    rng = np.random.default_rng(7)
    with B.from_config(c, 0, kernels=K, valid_yx=yx) as s:
        s.set_dm(modes)
        for T in (16, 3):
            ph = torch.from_numpy(W.phase_frames(c, 0, [t % 2 for t in range(T)])).cuda()
            coef = torch.from_numpy(rng.normal(0, 0.3, (T, M)).astype(np.float32)).cuda()
            finite(f"measure_residual T={T}", s.measure_residual(ph, coef), s.last_kernel)
        R = torch.from_numpy(rng.normal(0, 1e-3, (M, 2 * s.nsub)).astype(np.float32)).cuda()
        c0 = torch.zeros(M, device="cuda")
        sl, hist = s.closed_loop(ph, R, 0.3, c0)
        finite("closed_loop", sl, s.last_kernel)


def pyramid_cases():
    p = W.PYRAMIDS["tiny"]
    amp = W.pyramid_mask(p)
    ph = torch.from_numpy(W.pyramid_frames(p, range(2), 1.0)).cuda()
    for rep in range(2):
        with B.Pyrwfs(amp, p.Np, p.s, p.bp, p.r_mod, p.K, p.D_pix) as s:
            finite("pyramid tiny", s.measure(ph), "pyr_rows/cols/final/bin/signal")
            finite("pyramid quadrants", s.debug_quadrants(ph), "")


if __name__ == "__main__":
    torch.cuda.set_device(0)
    which = sys.argv[1:] or ["sensor", "lgs", "loop", "pyramid"]
    for w in which:
        {"sensor": sensor_cases, "lgs": lgs_cases, "loop": loop_cases, "pyramid": pyramid_cases}[w]()
    torch.cuda.synchronize()
    print("sanitizer workloads done")

"""Race and bounds evidence without a tool (compute-sanitizer is closed on this GPU pool, profiles/r02_sanitizer.md):

* every kernel family is run many times on the same input, alone and while another stream keeps the SMs and the
  memory system busy, and has to return bit-identical results -- a shared-memory or global-memory race shows up as
  a run-to-run difference (the kernels have no atomics on floating-point data, so they are deterministic by
  construction and any difference is a bug);
* outputs are written into the middle of a larger buffer whose guard bands must come back untouched;
* the same call on a buffer placed at the very end of a fresh allocation (a read past the last frame then runs
  off the allocation) must agree with the call on a roomy buffer.
-m gpu; goes through the C ABI like every parity test."""
import numpy as np
import pytest

from paper_1408_0698_b200 import workloads as W

pytestmark = pytest.mark.gpu

REPS = 40
GUARD = 4096            # floats on each side of an output


def _busy(torch, stream, seconds_hint=0.0):
    """Something unrelated that competes for SMs, L2 and DRAM on another stream."""
    a = torch.empty(64 << 20, dtype=torch.float32, device="cuda")
    with torch.cuda.stream(stream):
        for _ in range(6):
            a.normal_()
            a.mul_(1.0001)
    return a


def _guarded(torch, shape):
    n = int(np.prod(shape))
    buf = torch.full((n + 2 * GUARD,), -12345.0, dtype=torch.float32, device="cuda")
    return buf, buf[GUARD:GUARD + n].view(*shape)


def _check_guards(buf, n):
    assert bool((buf[:GUARD] == -12345.0).all()) and bool((buf[GUARD + n:] == -12345.0).all()), "guard band overwritten"


CASES = [  # (config, every n-th subaperture, frames, algorithm name, force the persistent instances)
    (1, 1, 4, "ALGO_WK", False), (1, 1, 4, "ALGO_AUTO", False), (1, 1, 4, "ALGO_LITERAL", False),
    (2, 3, 5, "ALGO_PRUNED_FFT", False), (2, 3, 5, "ALGO_WK", False),
    (3, 4, 37, "ALGO_WK", False), (3, 4, 3, "ALGO_AUTO", False), (3, 40, 3, "ALGO_WK_GENERIC", False),
    (5, 4, 9, "ALGO_WK_FFT", True), (5, 4, 9, "ALGO_WK_FFT", False),
]


@pytest.mark.parametrize("cfg_id,every,T,algo,persistent", CASES)
def test_sensor_kernels_are_deterministic_and_stay_in_bounds(gpu, monkeypatch, cfg_id, every, T, algo, persistent):
    torch, B = gpu
    if persistent:
        monkeypatch.setenv("SHWFS_FORCE_PERSISTENT", "1")     # read at shwfs_create
    else:
        monkeypatch.delenv("SHWFS_FORCE_PERSISTENT", raising=False)
    c = W.CONFIGS[cfg_id]
    with B.from_config(c, 0, kernels=None) as probe:
        yx = probe.valid_yx[::every].copy()
    K = W.elongation_kernels(c, 0, yx)
    ph_np = W.phase_frames(c, 0, [t % 3 for t in range(T)])
    # the frames sit at the very end of their allocation
    ph = torch.empty(ph_np.size, dtype=torch.float32, device="cuda")
    ph.copy_(torch.from_numpy(ph_np).reshape(-1))
    ph = ph.view(T, c.N, c.N)
    side = torch.cuda.Stream()
    with B.from_config(c, 0, kernels=K, valid_yx=yx) as s:
        s.algorithm = getattr(B, algo)
        buf, out = _guarded(torch, (T, s.nsub, 2))
        ref = s.measure(ph).clone()
        names = {s.last_kernel}
        assert bool(torch.isfinite(ref).all())
        for rep in range(REPS):
            keep = _busy(torch, side) if rep % 4 == 0 else None
            out.fill_(float("nan"))                 # a spot the deal skipped would otherwise keep its old value
            s.measure(ph, out=out)
            assert torch.equal(out, ref), (rep, s.last_kernel, int((out != ref).sum()))
            del keep
        names.add(s.last_kernel)
        _check_guards(buf, out.numel())
        if persistent:
            assert any("tma" in k for k in names), names
        # the binned debug image: same kernels with the image store on
        ibuf, img = _guarded(torch, (T, s.nsub, s.D, s.D))
        B.load().shwfs_debug_spots(s._h, ph.data_ptr(), T, 2, img.data_ptr(), None)
        torch.cuda.synchronize()
        _check_guards(ibuf, img.numel())
        assert torch.equal(img, s.debug_spots(ph, 2))


def test_lgs_and_loop_kernels_are_deterministic(gpu):
    """Multi-layer EXT instances with noise, the tcgen05 DM GEMM (hand-rolled mbarrier ring) and the closed loop."""
    torch, B = gpu
    c = W.CONFIGS[3]
    with B.from_config(c, 0, kernels=None) as probe:
        yx = probe.valid_yx[::6].copy()
    K = W.spot_size_kernels(c, yx)
    sod = W.sodium_layers(c, 0, 3)
    T, M = 33, 24
    ph = torch.from_numpy(W.phase_frames(c, 0, range(3))).cuda().repeat(T, 1, 1)[:T * 3].view(T, 3, c.N, c.N).contiguous()
    side = torch.cuda.Stream()
    with B.from_config(c, 0, kernels=K, valid_yx=yx) as s:
        s.set_sodium(sod["weight"], sod["defocus"], sod["tilt_x"], sod["tilt_y"], (sod["cx"], sod["cy"]))
        s.set_noise(5.0, 3.0, 99)
        ref = s.measure(ph).clone()
        for rep in range(REPS // 2):
            keep = _busy(torch, side) if rep % 4 == 0 else None
            assert torch.equal(s.measure(ph), ref), (rep, s.last_kernel)
            del keep
    Ke = W.elongation_kernels(c, 0, yx)
    rng = np.random.default_rng(11)
    with B.from_config(c, 0, kernels=Ke, valid_yx=yx) as s:
        s.set_dm(torch.from_numpy(W.dm_modes(c, M)).cuda())
        ph1 = torch.from_numpy(W.phase_frames(c, 0, [t % 3 for t in range(T)])).cuda()
        coef = torch.from_numpy(rng.normal(0, 0.3, (T, M)).astype(np.float32)).cuda()
        buf, out = _guarded(torch, (T, s.nsub, 2))
        ref = s.measure_residual(ph1, coef).clone()
        for rep in range(REPS // 2):
            keep = _busy(torch, side) if rep % 4 == 0 else None
            out.fill_(float("nan"))
            s.measure_residual(ph1, coef, out=out)
            assert torch.equal(out, ref), rep
            del keep
        _check_guards(buf, out.numel())
        R = torch.from_numpy(rng.normal(0, 1e-3, (M, 2 * s.nsub)).astype(np.float32)).cuda()
        sl0, h0 = s.closed_loop(ph1[:8], R, 0.3, torch.zeros(M, device="cuda"))
        for rep in range(5):
            sl, h = s.closed_loop(ph1[:8], R, 0.3, torch.zeros(M, device="cuda"))
            assert torch.equal(sl, sl0) and torch.equal(h, h0)


def test_pyramid_kernels_are_deterministic(gpu):
    torch, B = gpu
    p = W.PYRAMIDS["tiny"]
    amp = W.pyramid_mask(p)
    ph = torch.from_numpy(W.pyramid_frames(p, range(3), 1.0)).cuda()
    side = torch.cuda.Stream()
    with B.Pyrwfs(amp, p.Np, p.s, p.bp, p.r_mod, p.K, p.D_pix) as s:
        ref = s.measure(ph).clone()
        for rep in range(REPS // 2):
            keep = _busy(torch, side) if rep % 4 == 0 else None
            assert torch.equal(s.measure(ph), ref), rep
            del keep

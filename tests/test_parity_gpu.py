"""GPU <-> oracle parity through the C ABI (run on the B200 box with -m gpu).

Tolerances are BASELINE.json:north_star's: per-subaperture intensities within 1e-4 of the spot peak,
slopes within 1e-3 detector pixel absolute.  Every input is seeded and synthetic
(paper_1408_0698_b200.workloads); every expected value comes from oracle/ on the same fp32 arrays.
"""
import numpy as np
import pytest

from paper_1408_0698_b200 import workloads as W

pytestmark = pytest.mark.gpu

SLOPE_TOL = 1e-3      # detector px, absolute          (north_star)
IMAGE_TOL = 1e-4      # fraction of the spot peak      (north_star)


def _algos(sensor, B):
    out = []
    for a in (B.ALGO_WK, B.ALGO_WK_GENERIC, B.ALGO_LITERAL, B.ALGO_PRUNED_FFT, B.ALGO_WK_FFT):
        try:
            sensor.algorithm = a
            out.append(a)
        except B.ShwfsError as e:
            assert e.code == B.SHWFS_EUNSUPPORTED
    return out


def _img_err(got, want):
    pk = want.max(axis=(-2, -1), keepdims=True)
    return float((np.abs(got - want) / pk).max())


@pytest.mark.parametrize("cfg_id,T", [(1, 4), (2, 3), (3, 3), (5, 2)])
def test_slopes_and_binned_images_match_oracle(gpu, oracle, cfg_id, T):
    """Every spot of T full frames, every algorithm that has an instance for the sizes (configs 1,2,3,5;
    config 4 is config 3 with six launch points, covered by test_config4_* below)."""
    torch, B = gpu
    c = W.CONFIGS[cfg_id]
    amp = W.pupil_mask(c)
    ph = W.phase_frames(c, 0, range(T))
    with B.from_config(c, 0) as s:
        yx = s.valid_yx
        np.testing.assert_array_equal(yx, oracle.valid_list(amp, c.n, c.min_illum))
        K = W.elongation_kernels(c, 0, yx)
        want, wimg = oracle.measure(ph, amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K, stage=2)
        phd = torch.from_numpy(ph).cuda()
        algos = _algos(s, B)
        assert B.ALGO_WK in algos
        for a in algos:
            s.algorithm = a
            got = s.measure(phd).cpu().numpy()
            img = s.debug_spots(phd, 2).cpu().numpy()
            assert got.shape == (T, len(yx), 2)
            assert np.abs(got - want).max() <= SLOPE_TOL, (a, np.abs(got - want).max())
            assert _img_err(img, wimg) <= IMAGE_TOL, (a, _img_err(img, wimg))


@pytest.mark.parametrize("cfg_id,T", [(1, 4), (2, 1), (3, 1), (5, 1)])
def test_unbinned_intensities_match_oracle(gpu, oracle, cfg_id, T):
    """north_star: "per-subaperture intensities within 1e-4 of the spot peak" -- the centred P x P intensity
    |DFT(e)|^2/P^2 (stage 0) and the centred image after the elongation convolution (stage 1) of every spot,
    produced by the literal FFT chain, against the oracle's O4/O6 and O5/O6 images."""
    torch, B = gpu
    c = W.CONFIGS[cfg_id]
    amp = W.pupil_mask(c)
    ph = W.phase_frames(c, 0, range(T))
    with B.from_config(c, 0) as s:
        yx = s.valid_yx
        if cfg_id == 5:                                   # 64x64 float64 images: keep a spread subset
            yx = yx[:: 4]
        K = W.elongation_kernels(c, 0, s.valid_yx)
    if K is not None and cfg_id == 5:
        K = K[:: 4]
    with B.Shwfs(amp, c.S, c.n, c.dx, W.LAMBDA_M, c.P, c.b, valid_yx=yx, threshold_frac=c.tau,
                 elong_kernels=K) as s:
        phd = torch.from_numpy(ph).cuda()
        for stage in (0, 1):
            want_sl, wimg = oracle.measure(ph, amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K, stage=stage)
            img = s.debug_spots(phd, stage).cpu().numpy()
            assert img.shape == (T, len(yx), c.P, c.P)
            assert _img_err(img, wimg) <= IMAGE_TOL, (stage, _img_err(img, wimg))
        s.algorithm = B.ALGO_LITERAL
        got = s.measure(phd).cpu().numpy()
        assert np.abs(got - want_sl).max() <= SLOPE_TOL


@pytest.mark.parametrize("wfs", [0, 5])
def test_config4_full_batch_sampled_spots(gpu, oracle, wfs):
    """The launch configuration bench.py times: config 4, one 100-frame batch of one WFS (463 200 spots in
    one launch); 3000 sampled (frame, subaperture) outputs are recomputed one by one by the oracle."""
    torch, B = gpu
    c = W.CONFIGS[4]
    amp = W.pupil_mask(c)
    dev = torch.device("cuda")
    phd = W.phase_frames_device(c, wfs, range(c.batch), dev)
    with B.from_config(c, wfs) as s:
        yx = s.valid_yx
        got = s.measure(phd)
        assert s.launch_count == 1
        torch.cuda.synchronize()
        got = got.cpu().numpy()
    assert np.isfinite(got).all()
    rng = np.random.default_rng(1234 + wfs)
    ts = np.sort(rng.choice(c.batch, size=6, replace=False))
    ts[0], ts[-1] = 0, c.batch - 1                       # first and last frame of the launch
    for t in ts:
        idx = np.sort(rng.choice(len(yx), size=500, replace=False))
        idx[0], idx[-1] = 0, len(yx) - 1                 # first and last CTA / ragged tail
        K = W.elongation_kernels(c, wfs, yx, subset=idx)
        frame = phd[int(t)].cpu().numpy()[None]
        want = oracle.measure(frame, amp, yx[idx], c.n, c.P, c.b, tau=c.tau, kernels=K)
        err = np.abs(got[t, idx] - want[0]).max()
        assert err <= SLOPE_TOL, (int(t), err)


def test_config4_properties_at_full_size(gpu):
    """Properties that hold at any size: a flat wavefront gives zero slopes on every subaperture of every WFS
    geometry (I1), and frames are independent (permuting frames permutes slopes bit for bit)."""
    torch, B = gpu
    c = W.CONFIGS[4]
    with B.from_config(c, 3) as s:
        flat = torch.zeros((2, c.N, c.N), dtype=torch.float32, device="cuda")
        flat[1] += 3.25                                   # piston
        sl = s.measure(flat).cpu().numpy()
        assert np.abs(sl).max() <= 2e-5
        ph = W.phase_frames_device(c, 3, range(5), torch.device("cuda"))
        a = s.measure(ph).cpu().numpy()
        perm = [3, 0, 4, 1, 2]
        b = s.measure(ph[perm].contiguous()).cpu().numpy()
        np.testing.assert_array_equal(a[perm], b)


@pytest.mark.parametrize("T", [1, 31, 33, 65])
def test_ragged_batch_sizes(gpu, oracle, T):
    """T not a multiple of the 32-spot CTA: spots straddle subapertures and the last CTA is partly empty."""
    torch, B = gpu
    c = W.CONFIGS[1]
    amp = W.pupil_mask(c)
    ph = W.phase_frames(c, 0, [t % 4 for t in range(T)])
    rng = np.random.default_rng(T)
    K = rng.random((80, c.P, c.P)).astype(np.float32)     # arbitrary (asymmetric) kernels: complex table
    with B.Shwfs(amp, c.S, c.n, c.dx, W.LAMBDA_M, c.P, c.b, threshold_frac=0.1, elong_kernels=K) as s:
        yx = s.valid_yx
        want = oracle.measure(ph, amp, yx, c.n, c.P, c.b, tau=0.1, kernels=K)
        for a in _algos(s, B):
            s.algorithm = a
            got = s.measure(torch.from_numpy(ph).cuda()).cpu().numpy()
            assert np.abs(got - want).max() <= SLOPE_TOL, (a, T)


def test_t_zero_is_a_noop(gpu):
    torch, B = gpu
    c = W.CONFIGS[1]
    with B.from_config(c, 0) as s:
        ph = torch.empty((0, c.N, c.N), dtype=torch.float32, device="cuda")
        out = s.measure(ph)
        assert out.shape == (0, s.nsub, 2)
        assert s.launch_count == 0


@pytest.mark.parametrize("n,P,b", [(8, 16, 1), (10, 32, 2), (16, 32, 2), (16, 64, 4), (8, 32, 2), (10, 16, 1),
                                   (6, 16, 2), (12, 32, 1), (5, 8, 1), (12, 32, 2), (14, 32, 2), (14, 64, 4),
                                   (12, 16, 1)])
def test_small_grids_all_sizes(gpu, oracle, n, P, b):
    """3x3 subapertures with a partially lit mask, explicit valid list (including a dark subaperture), random
    phases of several radians, with and without kernels, tau 0 and 0.1, both threshold modes."""
    torch, B = gpu
    S = 3
    N = S * n
    rng = np.random.default_rng(n * 1000 + P + b)
    amp = (rng.random((N, N)) > 0.2).astype(np.float32) * rng.uniform(0.5, 1.0, (N, N)).astype(np.float32)
    amp[:n, :n] = 0.0                                      # a dark subaperture: sum Wt == 0 => (0,0)
    yx = np.array([[sy, sx] for sy in range(S) for sx in range(S)], dtype=np.int32)
    ph = rng.normal(0, 3.0, (5, N, N)).astype(np.float32)
    D = P // b
    for use_k in (False, True):
        K = rng.random((len(yx), P, P)).astype(np.float32) if use_k else None
        for tau, mode in ((0.0, 0), (0.1, 0), (0.3, 1)):
            try:
                s = B.Shwfs(amp, S, n, 0.05, W.LAMBDA_M, P, b, valid_yx=yx, threshold_frac=tau,
                            threshold_mode=mode, phase_to_rad=0.7, elong_kernels=K)
            except B.ShwfsError as e:
                assert e.code == B.SHWFS_EUNSUPPORTED and (n > 32 or D > 32)
                continue
            with s:
                want, wimg = oracle.measure(ph, amp, yx, n, P, b, c_phi=np.float32(0.7), tau=tau, mode=mode,
                                            kernels=K, stage=2)
                phd = torch.from_numpy(ph).cuda()
                for a in _algos(s, B):
                    s.algorithm = a
                    got = s.measure(phd).cpu().numpy()
                    img = s.debug_spots(phd, 2).cpu().numpy()
                    lit = wimg.max(axis=(2, 3)) > 0
                    assert (got[~lit] == 0).all()
                    assert np.abs(img[~lit]).max() == 0
                    assert _img_err(img[lit], wimg[lit]) <= IMAGE_TOL, (a, use_k, tau, mode)
                    if mode == 0:
                        assert np.abs(got - want).max() <= SLOPE_TOL, (a, use_k, tau, mode)
                    else:
                        # hard mask: a pixel within rounding of the threshold may flip (reading A7); compare
                        # the spots whose pixels all stay clear of it, require the rest to be valid CoGs
                        m = wimg.max(axis=(2, 3), keepdims=True)
                        clear = (np.abs(wimg - tau * m) > 1e-5 * m).all(axis=(2, 3)) | ~lit
                        assert np.abs(got - want)[clear].max() <= SLOPE_TOL
                        assert clear.mean() > 0.9
                        assert np.abs(got).max() <= (D - 1) / 2


def test_invariants_on_device(gpu):
    """I1 flat, I2 integer tilt, I7 piston / 2*pi wraps at +-1000 rad, I8 negation, on the device path itself."""
    torch, B = gpu
    c = W.CONFIGS[3]
    dev = torch.device("cuda")
    with B.from_config(c, 0) as s:
        ph = W.phase_frames_device(c, 0, range(1), dev)
        base = s.measure(ph).cpu().numpy()
        # I7: piston and integer multiples of 2*pi (range reduction at large arguments)
        k2pi = torch.randint(-150, 150, ph.shape, device=dev).to(torch.float64) * (2 * np.pi)
        wrapped = (ph.to(torch.float64) + k2pi).to(torch.float32)
        got = s.measure(wrapped).cpu().numpy()
        assert np.abs(got - base).max() <= 5e-3          # fp32 input rounding at |phi| ~ 1000 rad: ulp 6e-5 rad
        got = s.measure(ph + 1.0).cpu().numpy()
        assert np.abs(got - base).max() <= 1e-4
        # I8: phase negation reflects the spot about the detector centre: slopes negate
        neg = s.measure(-ph).cpu().numpy()
        assert np.abs(neg + base).max() <= 1e-4
        # I2: tilt by b unbinned pixels moves every centroid by exactly 1 detector px when nothing crosses the
        # edge; with wrapped elongated spots only check the un-elongated handle below
    c2 = W.CONFIGS[2]
    with B.from_config(c2, 0) as s:
        ph = 0.3 * W.phase_frames_device(c2, 0, range(1), dev)
        base = s.measure(ph).cpu().numpy()
        x = torch.arange(c2.N, device=dev, dtype=torch.float64)
        tilt = (2 * np.pi * c2.b / c2.P) * x[None, None, :]
        got = s.measure((ph.to(torch.float64) + tilt).to(torch.float32)).cpu().numpy()
        d = got - base
        keep = np.abs(base).max(axis=2) < 1.0             # well inside the field
        assert np.abs(d[keep][:, 0] - 1.0).max() <= 5e-2  # threshold keeps it near, not exactly, 1 (tails wrap)
        assert np.abs(d[keep][:, 1]).max() <= 5e-2


def test_nan_stays_in_its_spot(gpu):
    torch, B = gpu
    c = W.CONFIGS[1]
    with B.from_config(c, 0) as s:
        ph = torch.from_numpy(W.phase_frames(c, 0, range(2))).cuda()
        base = s.measure(ph).cpu().numpy()
        yx = s.valid_yx
        sy, sx = yx[7]
        ph2 = ph.clone()
        ph2[1, sy * c.n + 2, sx * c.n + 3] = float("nan")
        got = s.measure(ph2).cpu().numpy()
        mask = np.ones(got.shape[:2], bool)
        mask[1, 7] = False
        np.testing.assert_array_equal(got[mask], base[mask])


@pytest.mark.parametrize("pinned", [True, False])
def test_host_pipeline_copies_only_valid_runs(gpu, oracle, pinned):
    """shwfs_measure_host moves only the column runs of valid subapertures (strided 3-D copies): bit-identical
    to the device path on config 3 (annular pupil: two runs per lenslet row across the obstruction), from pinned
    and from pageable memory, with NaN planted everywhere outside the valid subapertures of the host frames."""
    torch, B = gpu
    c = W.CONFIGS[3]
    T = 30                                                    # 26-frame chunks: two chunks
    ph = W.phase_frames(c, 0, [t % 3 for t in range(T)])
    with B.from_config(c, 0) as s:
        yx = s.valid_yx
        lo = {sy: yx[yx[:, 0] == sy, 1].min() for sy in np.unique(yx[:, 0])}
        hi = {sy: yx[yx[:, 0] == sy, 1].max() for sy in np.unique(yx[:, 0])}
        assert s.host_bytes_per_frame == 4 * c.n * c.n * sum(hi[sy] - lo[sy] + 1 for sy in lo)
        assert s.host_bytes_per_frame < 0.82 * 4 * c.N * c.N
        dev = s.measure(torch.from_numpy(ph).cuda()).cpu().numpy()
        keep = np.zeros((c.N, c.N), bool)
        for sy in lo:                                          # the bounding extent of each lenslet row
            keep[sy * c.n:(sy + 1) * c.n, lo[sy] * c.n:(hi[sy] + 1) * c.n] = True
        poisoned = ph.copy()
        poisoned[:, ~keep] = np.nan
        if pinned:
            src = torch.from_numpy(poisoned).pin_memory()
            got = s.measure_host(src).numpy()
        else:
            got = s.measure_host(poisoned)
        np.testing.assert_array_equal(got, dev)
    c1 = W.CONFIGS[1]
    with B.from_config(c1, 0) as s:                            # 80 of 100 subapertures: still worth it
        assert s.host_bytes_per_frame == 4 * 80 * c1.n * c1.n    # no obstruction: the row extents hold valid patches only
        ph1 = W.phase_frames(c1, 0, range(4))
        np.testing.assert_array_equal(s.measure_host(ph1), s.measure(torch.from_numpy(ph1).cuda()).cpu().numpy())


@pytest.mark.parametrize("cfg_id", [2, 5])
def test_full_batch_sampled_spots_other_configs(gpu, oracle, cfg_id):
    """Configs 2 (pruned-FFT path, no elongation) and 5 (n = 16, pad 64, 4x4 binning, elongation <= 6 arcsec) at
    BASELINE.json's full batch size, in the one-launch configuration bench.py --config uses: 1500 sampled
    (frame, subaperture) outputs recomputed one by one by the oracle."""
    torch, B = gpu
    c = W.CONFIGS[cfg_id]
    amp = W.pupil_mask(c)
    dev = torch.device("cuda")
    phd = W.phase_frames_device(c, 0, range(c.batch), dev)
    with B.from_config(c, 0) as s:
        yx = s.valid_yx
        got = s.measure(phd)
        assert s.launch_count == 1
        torch.cuda.synchronize()
        got = got.cpu().numpy()
    assert np.isfinite(got).all()
    rng = np.random.default_rng(77 + cfg_id)
    for t in (0, int(rng.integers(1, c.batch - 1)), c.batch - 1):
        idx = np.sort(rng.choice(len(yx), size=500, replace=False))
        idx[0], idx[-1] = 0, len(yx) - 1
        K = W.elongation_kernels(c, 0, yx, subset=idx)
        frame = phd[int(t)].cpu().numpy()[None]
        want = oracle.measure(frame, amp, yx[idx], c.n, c.P, c.b, tau=c.tau, kernels=K)
        err = np.abs(got[t, idx] - want[0]).max()
        assert err <= SLOPE_TOL, (cfg_id, int(t), err)


@pytest.mark.parametrize("cfg_id", [4, 5])
def test_all_six_wfs_frames_0_1_499_999_in_full(gpu, oracle, cfg_id):
    """SURVEY.md 8(d) parity subset for configs 4-5: all six WFS (six launch points, independent seeded
    screens), frames {0, 1, 499, 999} of the 1000-frame stream, EVERY spot (6 x 4 x 4632 = 111 168 per config)
    against the oracle on the numpy-recipe frames."""
    torch, B = gpu
    c = W.CONFIGS[cfg_id]
    amp = W.pupil_mask(c)
    yx = oracle.valid_list(amp, c.n, c.min_illum)
    frames = [0, 1, 499, 999]
    worst = 0.0
    for w in range(c.W):
        ph = W.phase_frames(c, w, frames)
        K = W.elongation_kernels(c, w, yx, device=torch.device("cuda")).cpu().numpy()
        want = oracle.measure(ph, amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K)
        with B.Shwfs(amp, c.S, c.n, c.dx, W.LAMBDA_M, c.P, c.b, valid_yx=yx, threshold_frac=c.tau, elong_kernels=K) as s:
            got = s.measure(torch.from_numpy(ph).cuda()).cpu().numpy()
        err = float(np.abs(got - want).max())
        worst = max(worst, err)
        assert err <= SLOPE_TOL, (cfg_id, w, err)
    assert worst <= 1e-4          # measured margin: two orders below the tolerance


def test_register_gather_instance_and_alignment_contract(gpu, oracle, monkeypatch):
    """Config 2 takes its patches by TMA; SHWFS_NO_TMA (read at shwfs_create) selects the register-gather instance
    of the same kernel, which must give the same slopes; the library says which instance ran (shwfs_last_kernel).
    Frames that are not 16-byte aligned are outside the contract of include/shwfs.h: SHWFS_EINVAL, nothing launched."""
    torch, B = gpu
    c = W.CONFIGS[2]
    amp = W.pupil_mask(c)
    T = 2
    ph = W.phase_frames(c, 0, range(T))
    phd = torch.from_numpy(ph).cuda()
    want = None
    for no_tma, kind in ((False, "tma"), (True, "ldg")):
        if no_tma:
            monkeypatch.setenv("SHWFS_NO_TMA", "1")
        else:
            monkeypatch.delenv("SHWFS_NO_TMA", raising=False)
        with B.from_config(c, 0) as s:
            if want is None:
                want = oracle.measure(ph, amp, s.valid_yx, c.n, c.P, c.b, tau=c.tau)
            got = s.measure(phd).cpu().numpy()
            assert s.last_kernel == f"pruned_fft_kernel<32,16,0,{kind}>", s.last_kernel
            assert np.abs(got - want).max() <= SLOPE_TOL, (kind, np.abs(got - want).max())
            buf = torch.zeros(ph.size + 4, dtype=torch.float32, device="cuda")
            out = torch.empty((T, s.nsub, 2), dtype=torch.float32, device="cuda")
            n0 = s.launch_count
            for shift in (1, 2):
                view = buf[shift:shift + ph.size]
                assert view.data_ptr() % 16 != 0
                rc = B.load().shwfs_measure(s._h, view.data_ptr(), T, out.data_ptr(), None)
                assert rc == B.SHWFS_EINVAL
            assert s.launch_count == n0


def test_dynamic_deal_ragged_tails_match_oracle(gpu, oracle, monkeypatch):
    """The persistent instances deal chunks of consecutive spots to warps from a counter (csrc/sweep.cuh).  Totals
    that are odd, not a multiple of the chunk, smaller than one chunk per warp, and two calls back to back on one
    handle (the last warp re-arms the counter): every spot against the oracle.
    config 5 geometry (wkf_kernel<16,..,tma>, chunks of 16) on a subset of subapertures with the persistent instance
    forced; config 2 (pruned_fft_kernel<32,16,..,tma>, chunks of 4) at a size that takes the dynamic deal by itself."""
    torch, B = gpu
    monkeypatch.setenv("SHWFS_FORCE_PERSISTENT", "1")
    c = W.CONFIGS[5]
    amp = W.pupil_mask(c)
    full = oracle.valid_list(amp, c.n, c.min_illum)
    yx = full[::7][:661].copy()
    K = W.elongation_kernels(c, 0, yx)
    with B.from_config(c, 0, kernels=K, valid_yx=yx) as s:
        for T in (3, 1, 3):
            ph = W.phase_frames(c, 0, range(T))
            assert (T * len(yx)) % 2 == 1
            want = oracle.measure(ph, amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K)
            out = torch.full((T, len(yx), 2), float("nan"), dtype=torch.float32, device="cuda")   # skipped spot = NaN
            got = s.measure(torch.from_numpy(ph).cuda(), out=out).cpu().numpy()
            assert s.last_kernel == "wkf_kernel<16,0,0,tma>", s.last_kernel
            assert np.abs(got - want).max() <= SLOPE_TOL, (T, np.abs(got - want).max())
    monkeypatch.delenv("SHWFS_FORCE_PERSISTENT")
    c = W.CONFIGS[2]
    amp = W.pupil_mask(c)
    yx = oracle.valid_list(amp, c.n, c.min_illum)[:1211].copy()
    T = 17
    ph = W.phase_frames(c, 0, [t % 4 for t in range(T)])
    assert (T * len(yx)) % 4 == 3 and T * len(yx) >= 4 * 8 * 4 * 148
    want = oracle.measure(ph[:4], amp, yx, c.n, c.P, c.b, tau=c.tau)
    with B.from_config(c, 0, valid_yx=yx) as s:
        phd = torch.from_numpy(ph).cuda()
        for rep in range(2):
            out = torch.full((T, len(yx), 2), float("nan"), dtype=torch.float32, device="cuda")
            got = s.measure(phd, out=out).cpu().numpy()
            assert s.last_kernel == "pruned_fft_kernel<32,16,0,tma>"
            for t in range(T):
                assert np.abs(got[t] - want[t % 4]).max() <= SLOPE_TOL, (rep, t)

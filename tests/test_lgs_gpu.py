"""GPU <-> oracle parity of the paper's full LGS model through the C ABI (run on the B200 box, -m gpu):
sodium sub-layer sum (shwfs_set_sodium) and detector noise (shwfs_set_noise, f2),
PAPER.md:85-87, 91.  Tolerances are north_star's (images 1e-4 of the spot peak, slopes 1e-3 px); every
expected value comes from oracle/shwfs_oracle_lgs.c on the same seeded fp32 inputs."""
import numpy as np
import pytest

from paper_1408_0698_b200 import workloads as W

pytestmark = pytest.mark.gpu

SLOPE_TOL = 1e-3
IMAGE_TOL = 1e-4


def _img_err(got, want):
    pk = want.max(axis=(-2, -1), keepdims=True)
    return float((np.abs(got - want) / pk).max())


def _wk_algos(s, B):
    out = []
    for a in (B.ALGO_WK, B.ALGO_WK_GENERIC, B.ALGO_WK_FFT):
        try:
            s.algorithm = a
            out.append(a)
        except B.ShwfsError as e:
            assert e.code == B.SHWFS_EUNSUPPORTED
    return out


@pytest.mark.parametrize("L,shared", [(3, False), (5, True)])
def test_config3_sublayers_match_oracle(gpu, oracle, L, shared):
    """MAORY single-LGS geometry (config 3: 4632 subapertures of 10x10 px, pad 32, 2x2 binning, tau 0.1) with
    L sodium sub-layers (workloads.sodium_layers: Gaussian profile, defocus about the launch point, uplink
    tilts), round 1-arcsec spot-size kernel; every spot of 2 time steps."""
    torch, B = gpu
    c = W.CONFIGS[3]
    amp = W.pupil_mask(c)
    T = 2
    sod = W.sodium_layers(c, 0, L)
    if shared:
        ph = W.phase_frames(c, 0, range(T))
    else:
        ph = np.stack([W.phase_frames(c, 0, range(10 * l, 10 * l + T)) for l in range(L)], axis=1)
    yx = oracle.valid_list(amp, c.n, c.min_illum)
    K = W.spot_size_kernels(c, yx)
    want, wimg = oracle.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, weight=sod["weight"], defocus=sod["defocus"],
                                    tilt_x=sod["tilt_x"], tilt_y=sod["tilt_y"], cx=sod["cx"], cy=sod["cy"],
                                    tau=c.tau, kernels=K, stage=2)
    with B.from_config(c, 0, kernels=K, valid_yx=yx) as s:
        s.set_sodium(sod["weight"], sod["defocus"], sod["tilt_x"], sod["tilt_y"], (sod["cx"], sod["cy"]),
                     shared_phase=shared)
        phd = torch.from_numpy(ph).cuda()
        for a in _wk_algos(s, B):
            s.algorithm = a
            l0 = s.launch_count
            got = s.measure(phd).cpu().numpy()
            assert s.launch_count == l0 + 1                     # all sub-layers in ONE launch
            img = s.debug_spots(phd, 2).cpu().numpy()
            assert np.abs(got - want).max() <= SLOPE_TOL, (a, np.abs(got - want).max())
            assert _img_err(img, wimg) <= IMAGE_TOL, (a, _img_err(img, wimg))
        # back to the single-layer sensor
        s.set_sodium(None)
        one = s.measure(torch.from_numpy(np.ascontiguousarray(ph[:, 0] if not shared else ph)).cuda()).cpu().numpy()
        ref = oracle.measure(ph[:, 0] if not shared else ph, amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K)
        assert np.abs(one - ref).max() <= SLOPE_TOL


def test_config3_noise_matches_oracle(gpu, oracle):
    """Detector noise (photon + read, Philox4x32-10) on the sub-layer image: the noisy image and the slopes
    against the oracle for every spot; first_frame continues the noise stream across calls."""
    torch, B = gpu
    c = W.CONFIGS[3]
    amp = W.pupil_mask(c)
    T, L = 3, 3
    sod = W.sodium_layers(c, 0, L)
    ph = W.phase_frames(c, 0, range(T))
    yx = oracle.valid_list(amp, c.n, c.min_illum)
    K = W.spot_size_kernels(c, yx)
    F, ron, seed = 500.0 / c.n ** 2, 3.0, 0x1408069800000091
    kw = dict(weight=sod["weight"], defocus=sod["defocus"], tilt_x=sod["tilt_x"], tilt_y=sod["tilt_y"],
              cx=sod["cx"], cy=sod["cy"], tau=c.tau, kernels=K)
    want, wimg = oracle.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, flux=F, ron=ron, seed=seed, stage=3, **kw)
    clean = oracle.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, **kw)
    assert np.abs(want - clean).max() > 0.05                     # the noise does move the centroids
    with B.from_config(c, 0, kernels=K, valid_yx=yx) as s:
        s.set_sodium(sod["weight"], sod["defocus"], sod["tilt_x"], sod["tilt_y"], (sod["cx"], sod["cy"]),
                     shared_phase=True)
        s.set_noise(F, ron, seed)
        phd = torch.from_numpy(ph).cuda()
        for a in _wk_algos(s, B):
            s.algorithm = a
            got = s.measure(phd).cpu().numpy()
            img = s.debug_spots(phd, 3).cpu().numpy()
            assert _img_err(img, wimg) <= IMAGE_TOL, (a, _img_err(img, wimg))
            assert np.abs(got - want).max() <= SLOPE_TOL, (a, np.abs(got - want).max())
        # noise on the plain single-layer sensor (no sodium model set)
        s.set_sodium(None)
        w1, i1 = oracle.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, weight=[1.0], defocus=[0.0], tau=c.tau,
                                    kernels=K, flux=F, ron=ron, seed=seed, stage=3)
        for a in _wk_algos(s, B):
            s.algorithm = a
            got = s.measure(phd).cpu().numpy()
            img = s.debug_spots(phd, 3).cpu().numpy()
            assert _img_err(img, i1) <= IMAGE_TOL, (a, _img_err(img, i1))
            assert np.abs(got - w1).max() <= SLOPE_TOL, (a, np.abs(got - w1).max())
        s.set_sodium(sod["weight"], sod["defocus"], sod["tilt_x"], sod["tilt_y"], (sod["cx"], sod["cy"]),
                     shared_phase=True)
        s.algorithm = B.ALGO_WK
        # frames 1.. of the same stream in a second call
        s.set_noise(F, ron, seed, first_frame=1)
        tail = s.measure(phd[1:].contiguous()).cpu().numpy()
        assert np.abs(tail - want[1:]).max() <= SLOPE_TOL
        # another seed gives other noise; flux 0 switches it off
        s.set_noise(F, ron, seed + 1)
        other = s.measure(phd).cpu().numpy()
        assert np.abs(other - want).max() > 0.05
        s.set_noise(0.0)
        off = s.measure(phd).cpu().numpy()
        assert np.abs(off - clean).max() <= SLOPE_TOL


@pytest.mark.parametrize("n,P,b", [(8, 16, 1), (10, 32, 2), (16, 64, 4), (16, 32, 2), (6, 16, 1), (12, 32, 2),
                                   (14, 32, 2)])
def test_small_grids_sublayers_and_noise(gpu, oracle, n, P, b):
    """3x3 subapertures, partially lit mask with a dark subaperture, random kernels, 1..4 sub-layers with
    large random defocus / tilts (several wraps per patch), own or shared wavefronts, with and without
    noise, both threshold modes, specialised and generic kernels."""
    torch, B = gpu
    S, N, dx = 3, 3 * n, 0.05
    rng = np.random.default_rng(100 * n + P + b)
    amp = (rng.random((N, N)) > 0.2).astype(np.float32) * rng.uniform(0.5, 1.0, (N, N)).astype(np.float32)
    amp[:n, :n] = 0.0
    yx = np.array([[sy, sx] for sy in range(S) for sx in range(S)], dtype=np.int32)
    K = rng.random((len(yx), P, P)).astype(np.float32)
    T = 5
    for L, shared, tau, mode, F in ((1, True, 0.0, 0, 0.0), (2, False, 0.1, 0, 0.0), (4, False, 0.1, 0, 30.0),
                                    (3, True, 0.2, 1, 0.0), (1, False, 0.1, 0, 30.0)):
        ph = rng.normal(0, 2.0, (T, N, N) if shared else (T, L, N, N)).astype(np.float32)
        w = rng.uniform(0.1, 1.0, L)
        de = rng.normal(0, 40.0, L)                      # rad/m^2: up to ~20 rad across the 3n-pixel pupil
        tx, ty = rng.normal(0, 60.0, (2, L))             # rad/m: several rad per pixel
        cx, cy = 0.11, -0.23
        kw = dict(weight=w, defocus=de, tilt_x=tx, tilt_y=ty, cx=cx, cy=cy, tau=tau, mode=mode, kernels=K,
                  c_phi=np.float32(0.7), flux=F, ron=1.5, seed=42)
        want, wimg = oracle.measure_lgs(ph, amp, yx, n, P, b, dx, stage=3, **kw)
        with B.Shwfs(amp, S, n, dx, W.LAMBDA_M, P, b, valid_yx=yx, threshold_frac=tau, threshold_mode=mode,
                     phase_to_rad=0.7, elong_kernels=K) as s:
            s.set_sodium(w, de, tx, ty, (cx, cy), shared_phase=shared)
            s.set_noise(F, 1.5, 42)
            phd = torch.from_numpy(ph).cuda()
            algos = _wk_algos(s, B)
            assert B.ALGO_WK_GENERIC in algos
            for a in algos:
                s.algorithm = a
                got = s.measure(phd).cpu().numpy()
                img = s.debug_spots(phd, 3).cpu().numpy()
                lit = wimg.max(axis=(2, 3)) > 0
                if F == 0.0:
                    assert (got[~lit] == 0).all()
                assert _img_err(img[lit], wimg[lit]) <= IMAGE_TOL, (a, L, shared, F)
                if mode == 0:
                    sel = lit if F == 0.0 else np.ones_like(lit)
                    assert np.abs(got - want)[sel].max() <= SLOPE_TOL, (a, L, shared, F)
                else:
                    m = wimg.max(axis=(2, 3), keepdims=True)
                    clear = (np.abs(wimg - tau * m) > 1e-5 * m).all(axis=(2, 3)) | ~lit
                    assert np.abs(got - want)[clear].max() <= SLOPE_TOL
                    assert clear.mean() > 0.9


def test_host_pipeline_with_sublayers_and_noise(gpu, oracle):
    """shwfs_measure_host with [T,L,N,N] input cut into several chunks: identical (bit for bit) to one device
    call -- the chunks carry their frame offset into the noise counters -- and within tolerance of the oracle."""
    torch, B = gpu
    c = W.CONFIGS[1]
    amp = W.pupil_mask(c)
    L, T = 2, 300                                         # 256-frame chunks = 128 time steps: 3 chunks
    rng = np.random.default_rng(7)
    base = W.phase_frames(c, 0, range(4))
    ph = np.ascontiguousarray(base[rng.integers(0, 4, (T, L))] * rng.uniform(0.5, 1.5, (T, L, 1, 1)).astype(np.float32))
    with B.from_config(c, 0) as s:
        yx = s.valid_yx
        w, de = np.array([0.7, 0.3]), np.array([0.4, -0.6])
        s.set_sodium(w, de, None, None, (4.0, 0.0))
        s.set_noise(20.0, 2.0, 99, first_frame=5)
        dev = s.measure(torch.from_numpy(ph).cuda()).cpu().numpy()
        host = s.measure_host(ph)
        np.testing.assert_array_equal(host, dev)
        sub = [0, 127, 128, 299]
        want = np.stack([oracle.measure_lgs(ph[t:t + 1], amp, yx, c.n, c.P, c.b, c.dx, weight=w, defocus=de,
                                            cx=4.0, cy=0.0, tau=c.tau, flux=20.0, ron=2.0, seed=99)[0]
                         for t in sub])
        # the oracle's frame index is the index inside its call: recompute with the right counters instead
        for k, t in enumerate(sub):
            _, b2 = oracle.measure_lgs(ph[t:t + 1], amp, yx, c.n, c.P, c.b, c.dx, weight=w, defocus=de, cx=4.0,
                                       cy=0.0, tau=c.tau, stage=2)
            for i in (0, len(yx) - 1):
                noisy = oracle.add_noise(b2[0, i], 20.0, 2.0, 99, 5 + t, i)
                assert np.abs(dev[t, i] - oracle.threshold_cog(noisy, c.tau, 0)).max() <= SLOPE_TOL
        assert want.shape == (4, len(yx), 2)


def test_sodium_and_noise_argument_checking(gpu):
    torch, B = gpu
    c = W.CONFIGS[1]
    with B.from_config(c, 0) as s:
        for bad in (dict(weight=[-1.0], defocus=[0.0]), dict(weight=[np.nan], defocus=[0.0]),
                    dict(weight=[1.0] * 9, defocus=[0.0] * 9), dict(weight=[1.0], defocus=[np.inf])):
            with pytest.raises(B.ShwfsError) as e:
                s.set_sodium(**bad)
            assert e.value.code == B.SHWFS_EINVAL
        with pytest.raises(B.ShwfsError) as e:
            s.set_noise(10.0, -1.0)
        assert e.value.code == B.SHWFS_EINVAL
        s.set_sodium([1.0], [0.0])                        # a plain layer: same as the single-layer sensor
        ph = torch.from_numpy(W.phase_frames(c, 0, range(2))).cuda()
        a = s.measure(ph).cpu().numpy()
        s.set_sodium(None)
        s.algorithm = B.ALGO_WK
        b = s.measure(ph).cpu().numpy()
        assert np.abs(a - b).max() <= 1e-5
        with pytest.raises(B.ShwfsError) as e:            # stages 0/1 exist only for the single-layer sensor
            s.set_sodium([0.5, 0.5], [0.1, -0.1], shared_phase=True)
            s.debug_spots(ph, 0)
        assert e.value.code == B.SHWFS_EUNSUPPORTED
    # a size with no lag-domain instance (D = 64): literal chain only -> EUNSUPPORTED
    n, P = 8, 64
    amp = np.ones((2 * n, 2 * n), np.float32)
    with B.Shwfs(amp, 2, n, 0.1, W.LAMBDA_M, P, 1) as s:
        assert s.algorithm == B.ALGO_LITERAL
        with pytest.raises(B.ShwfsError) as e:
            s.set_sodium([1.0], [0.0])
        assert e.value.code == B.SHWFS_EUNSUPPORTED
        with pytest.raises(B.ShwfsError) as e:
            s.set_noise(10.0, 1.0)
        assert e.value.code == B.SHWFS_EUNSUPPORTED


# margin below which a Poisson draw may legitimately come out differently in fp32.  The device's rate F*B differs
# from the oracle's by ~2e-6 of the spot's peak rate (the measured image error; the tolerance is 1e-4), i.e. by
# d = 2e-6 x rate at the bright pixels.  In the inversion branch that moves every CDF value by at most d x pmf
# < 1e-5; in the rejection branch it moves the argument of the floor by d itself.  Clear = decided by more than
# 1e-4 + 1e-5 x rate (five times the measured error; the fp32 search itself adds ~1e-6).
def _poisson_clear(margin, rate):
    return margin > 1e-4 + 1e-5 * rate


@pytest.mark.parametrize("flux_total,ron", [(300.0, 0.0), (300.0, 3.0), (40000.0, 2.0)])
def test_config3_poisson_noise_matches_oracle(gpu, oracle, flux_total, ron):
    """photon_model = 1 (SURVEY.md 8(f) f2 as written: Poisson photon noise + Gaussian read noise).  The counts
    are integers decided by floating-point comparisons, so the statement is the one of the hard-mask threshold
    test: on every pixel whose draw was decided by a margin larger than rounding (_poisson_clear; the oracle
    reports the margin of each draw) the device count equals the oracle's exactly (with read noise: to 1e-4 of the peak);
    on spots whose 256 pixels are all clear the slopes agree to 1e-3 px; the remaining pixels differ by at most
    one count (inversion, rate < 30) or stay within 8 sigma of the rate (rejection branch, where a flipped
    acceptance moves on to the next attempt).  300 e-/subaperture exercises the inversion branch, 40000 the
    transformed rejection."""
    torch, B = gpu
    c = W.CONFIGS[3]
    amp = W.pupil_mask(c)
    T = 2
    ph = W.phase_frames(c, 0, range(T))
    yx = oracle.valid_list(amp, c.n, c.min_illum)[::3].copy()
    K = W.elongation_kernels(c, 0, yx)
    F, seed = flux_total / c.n ** 2, 0x14080698000000A7
    kw = dict(weight=[1.0], defocus=[0.0], tau=c.tau, kernels=K, flux=F, ron=ron, seed=seed, photon_model=1)
    want, wimg, margin = oracle.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, stage=3, want_margins=True, **kw)
    _, clean_img = oracle.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, weight=[1.0], defocus=[0.0], tau=c.tau,
                                      kernels=K, stage=2)
    rate = np.maximum(F * clean_img, 0.0)
    assert (rate >= 30).any() == (flux_total > 1000)                  # which branch the case exercises
    clear = _poisson_clear(margin, rate)
    bright = flux_total > 1000            # rates of thousands: the clearance 1e-5 x rate is a few percent of a count
    assert clear.mean() > (0.95 if bright else 0.99), clear.mean()
    spot_clear = clear.all(axis=(2, 3))
    assert bright or spot_clear.mean() > 0.3, spot_clear.mean()
    with B.from_config(c, 0, kernels=K, valid_yx=yx) as s:
        s.set_noise(F, ron, seed, photon_model=1)
        phd = torch.from_numpy(ph).cuda()
        for a in _wk_algos(s, B):
            s.algorithm = a
            got = s.measure(phd).cpu().numpy()
            img = s.debug_spots(phd, 3).cpu().numpy().astype(np.float64)
            d = np.abs(img - wimg)
            if ron == 0.0:
                assert np.all(img == np.round(img)) and img.min() >= 0
                assert np.all(d[clear] == 0.0), (a, d[clear].max(), int((d[clear] > 0).sum()))
            else:
                pk = wimg.max(axis=(2, 3), keepdims=True)
                assert (d / pk)[clear].max() <= IMAGE_TOL, (a, (d / pk)[clear].max())
            low = ~clear & (rate < 29.9)
            assert d[low].max(initial=0.0) <= 1.0 + 1e-3, (a, d[low].max())
            high = ~clear & (rate >= 29.9)
            assert np.all(d[high] <= 8.0 * np.sqrt(rate[high]) + 2.0)
            # slopes: wherever the noisy image is the oracle's (every all-clear spot, and every other spot whose
            # unclear draws happened to fall the same way), the centroid is the oracle's
            same = (d <= (1e-6 if ron == 0.0 else IMAGE_TOL * wimg.max(axis=(2, 3), keepdims=True))).all(axis=(2, 3))
            assert np.all(same[spot_clear]) and same.mean() > (0.05 if bright else 0.3), same.mean()
            assert np.abs(got - want)[same].max() <= SLOPE_TOL, (a, np.abs(got - want)[same].max())
            # elsewhere a handful of +-1 counts moves it by (lever arm / photo-electrons) each
            assert np.abs(got - want).max() <= (0.02 if bright else 0.5)
            # and the unclear pixels are as rare on the device as the margins say: no systematic disagreement
            assert (d > 0.5).mean() <= 2.0 * (~clear).mean() + 1e-4
        # the two models draw from one seed but are different noise; model 0 is unchanged by the new field
        s.algorithm = B.ALGO_WK
        s.set_noise(F, max(ron, 1.0), seed, photon_model=0)
        g0 = s.measure(phd).cpu().numpy()
        w0 = oracle.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, weight=[1.0], defocus=[0.0], tau=c.tau, kernels=K,
                                flux=F, ron=max(ron, 1.0), seed=seed)
        assert np.abs(g0 - w0).max() <= SLOPE_TOL
    with B.from_config(c, 0, kernels=K, valid_yx=yx) as s:
        nz = B.ShwfsNoise(1.0, 1.0, 1, 0, 2)
        import ctypes
        assert B.load().shwfs_set_noise(s._h, ctypes.byref(nz)) == B.SHWFS_EINVAL

"""GPU <-> oracle parity of the pyramid WFS (include/pyrwfs.h) through the C
ABI, -m gpu.  Tolerances: quadrant images within 1e-4 of their peak, signals within
2e-4 absolute (signals are dimensionless, |s| <~ 1)."""
import numpy as np
import pytest

from paper_1408_0698_b200 import workloads as W

pytestmark = pytest.mark.gpu

SIG_TOL = 2e-4
IMG_TOL = 1e-4


@pytest.fixture(scope="module")
def pyr():
    from oracle import pyramid
    return pyramid


@pytest.mark.parametrize("name,T,scale", [("tiny", 5, 1.0), ("lbt", 2, 0.3)])
def test_signals_and_quadrants_match_oracle(gpu, pyr, name, T, scale):
    torch, B = gpu
    p = W.PYRAMIDS[name]
    amp = W.pyramid_mask(p)
    ph = W.pyramid_frames(p, range(T), scale)
    yx = pyr.valid_pixels(amp, p.bp)
    want, wq = pyr.measure(ph, amp, yx, p.Np, p.s, p.bp, p.r_mod, p.K, p.D_pix, return_quadrants=True)
    with B.Pyrwfs(amp, p.Np, p.s, p.bp, p.r_mod, p.K, p.D_pix) as s:
        np.testing.assert_array_equal(s.valid_yx, yx)
        phd = torch.from_numpy(ph).cuda()
        got = s.measure(phd).cpu().numpy()
        q = s.debug_quadrants(phd).cpu().numpy()
        assert got.shape == want.shape
        assert np.abs(q - wq).max() <= IMG_TOL * wq.max(), np.abs(q - wq).max() / wq.max()
        assert np.abs(got - want).max() <= SIG_TOL, np.abs(got - want).max()


@pytest.mark.parametrize("N,Np,s,bp,r_mod,K", [(32, 256, 64, 2, 0.0, 0), (100, 256, 64, 5, 2.0, 4), (128, 256, 64, 4, 5.0, 12),
                                               (60, 1024, 200, 3, 1.5, 6)])
def test_small_pupils_all_shapes(gpu, pyr, N, Np, s, bp, r_mod, K):
    """Partially transmitting random masks (no symmetry), several radians of random phase, unmodulated and
    modulated, N not a multiple of the 8-line CTA, phase_to_rad != 1, ragged frame counts."""
    torch, B = gpu
    rng = np.random.default_rng(N + Np + K)
    ax = np.arange(N) + 0.5 - N / 2
    amp = ((np.hypot(ax[None, :], ax[:, None]) <= N / 2) * rng.uniform(0.4, 1.0, (N, N))).astype(np.float32)
    ph = rng.normal(0, 2.0, (3, N, N)).astype(np.float32)
    yx = pyr.valid_pixels(amp, bp, 0.3)
    want, wq = pyr.measure(ph, amp, yx, Np, s, bp, r_mod, K, 0.9 * N, c_phi=np.float32(0.6), return_quadrants=True)
    with B.Pyrwfs(amp, Np, s, bp, r_mod, K, 0.9 * N, min_illum=0.3, phase_to_rad=0.6) as sn:
        phd = torch.from_numpy(ph).cuda()
        got = sn.measure(phd).cpu().numpy()
        q = sn.debug_quadrants(phd).cpu().numpy()
        assert np.abs(q - wq).max() <= IMG_TOL * wq.max()
        assert np.abs(got - want).max() <= SIG_TOL


def test_tilt_response_and_flat_symmetry_on_device(gpu):
    """V4/V5 on the device path itself: flat wavefront -> antisymmetric s_x, zero mean; a tilt of 1 lambda/D
    under 4 lambda/D modulation -> mean s_x near (2/pi) asin(1/4)."""
    torch, B = gpu
    N, Np, s, bp = 64, 256, 64, 2
    ax = np.arange(N) + 0.5 - N / 2
    amp = (np.hypot(ax[None, :], ax[:, None]) <= N / 2).astype(np.float32)
    x = np.arange(N, dtype=np.float64)
    tilt = np.broadcast_to(2 * np.pi * x[None, :] / N, (N, N)).astype(np.float32)
    with B.Pyrwfs(amp, Np, s, bp, 4.0, 32, float(N)) as sn:
        ph = torch.from_numpy(np.stack([np.zeros((N, N), np.float32), tilt])).cuda()
        sig = sn.measure(ph).cpu().numpy()
        yx = sn.valid_yx
        Sp = N // bp
        grid = np.full((Sp, Sp), np.nan); grid[yx[:, 0], yx[:, 1]] = sig[0, :, 0]
        np.testing.assert_allclose(grid[:, ::-1], -grid, atol=2e-5, equal_nan=True)
        assert abs(sig[0].mean()) < 1e-5
        assert sig[1, :, 0].mean() == pytest.approx((2 / np.pi) * np.arcsin(0.25), rel=0.12)
        assert abs(sig[1, :, 1].mean()) < 5e-3


def test_chunking_and_argument_checking(gpu, pyr):
    torch, B = gpu
    p = W.PYRAMIDS["tiny"]
    amp = W.pyramid_mask(p)
    with B.Pyrwfs(amp, p.Np, p.s, p.bp, p.r_mod, p.K, p.D_pix) as s:
        T = 70                                            # more than one 64-frame chunk
        ph = torch.from_numpy(W.pyramid_frames(p, [t % 3 for t in range(T)])).cuda()
        a = s.measure(ph).cpu().numpy()
        np.testing.assert_array_equal(a[0], a[3]); np.testing.assert_array_equal(a[1], a[67])
        assert s.measure(ph[:0]).shape == (0, s.nvalid, 2)
    for kw, code in ((dict(pad=512), B.SHWFS_EUNSUPPORTED), (dict(pad=300), B.SHWFS_EINVAL),
                     (dict(separation=10), B.SHWFS_EINVAL), (dict(separation=120), B.SHWFS_EINVAL),
                     (dict(bin=5), B.SHWFS_EINVAL), (dict(pupil_diameter_px=0.0), B.SHWFS_EINVAL)):
        args = dict(pad=p.Np, separation=p.s, bin=p.bp, mod_radius=p.r_mod, mod_points=p.K, pupil_diameter_px=p.D_pix)
        args.update(kw)
        with pytest.raises(B.ShwfsError) as e:
            B.Pyrwfs(amp, **args)
        assert e.value.code == code, kw

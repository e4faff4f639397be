"""Pins of the pyramid-WFS oracle (oracle/pyramid.py).  CPU only.

V1 the two numpy.fft steps against explicit exponential sums; V2 no pyramid, no modulation returns the pupil;
V3 energy is conserved through the unit-modulus mask; V4 symmetries of the flat-wavefront signal; V5 sign and
size of the tilt response against the geometric-optics law of a modulated pyramid (2/pi) asin(theta/r_mod);
V6 transposition swaps s_x and s_y; V7 modulation = mean over explicit tilts; V8 piston; V9 each face carries the light of one
focal-plane quadrant."""
import numpy as np
import pytest

rng = np.random.default_rng(92)


@pytest.fixture(scope="module")
def pyr():
    from oracle import pyramid
    return pyramid


def _disc(N, obstruction=0.0):
    ax = np.arange(N) + 0.5 - N / 2
    r = np.hypot(ax[None, :], ax[:, None])
    return ((r <= N / 2) & (r >= obstruction * N / 2)).astype(np.float32)


def test_V1_chain_against_explicit_sums(pyr):
    N, Np, s = 4, 8, 2
    amp = rng.uniform(0.5, 1, (N, N)).astype(np.float32)
    ph = rng.normal(0, 1, (N, N)).astype(np.float32)
    r_mod, th, D = 1.3, 0.7, 4.0
    e = pyr.field(ph, amp, Np, r_mod, th, D)
    # Q1 written out
    for (y, x) in ((0, 0), (2, 3), (3, 1)):
        want = amp[y, x] * np.exp(1j * (ph[y, x] + 2 * np.pi * r_mod * (x * np.cos(th) + y * np.sin(th)) / D))
        assert abs(e[y, x] - want) < 1e-14
    assert np.abs(e[N:, :]).max() == 0 and np.abs(e[:, N:]).max() == 0
    k = np.arange(Np)
    W = np.exp(-2j * np.pi * np.outer(k, k) / Np)
    F = W @ e @ W.T                                              # Q2: sum e[y,x] w^(vy + ux)
    us = np.where(k < Np // 2, k, k - Np)
    M = np.exp(-2j * np.pi * s * (np.abs(us)[None, :] + np.abs(us)[:, None]) / Np)
    G = np.conj(W) @ (F * M) @ np.conj(W).T / Np ** 2            # Q4
    I = pyr.detector_intensity(ph, amp, Np, s, 0.0, 0, D)
    e0 = pyr.field(ph, amp, Np, 0.0, 0.0, D)
    G0 = np.conj(W) @ ((W @ e0 @ W.T) * M) @ np.conj(W).T / Np ** 2
    np.testing.assert_allclose(I, np.abs(G0) ** 2, atol=1e-13)
    np.testing.assert_allclose(pyr.pyramid_mask(Np, s), M, atol=1e-15)
    assert np.abs(np.fft.ifft2(np.fft.fft2(e) * M) - G).max() < 1e-13


def test_V2_no_pyramid_returns_the_pupil(pyr):
    N, Np = 12, 32
    amp = _disc(N) * rng.uniform(0.5, 1, (N, N)).astype(np.float32)
    ph = rng.normal(0, 2, (N, N)).astype(np.float32)
    I = pyr.detector_intensity(ph, amp, Np, 0, 0.0, 0, N)
    want = np.zeros((Np, Np)); want[:N, :N] = amp.astype(np.float64) ** 2
    np.testing.assert_allclose(I, want, atol=1e-13)


@pytest.mark.parametrize("K,r_mod", [(0, 0.0), (8, 3.0)])
def test_V3_energy_is_conserved(pyr, K, r_mod):
    N, Np, s = 16, 64, 16
    amp = _disc(N, 0.3)
    ph = rng.normal(0, 1.5, (N, N)).astype(np.float32)
    I = pyr.detector_intensity(ph, amp, Np, s, r_mod, K, N)
    assert I.sum() == pytest.approx((amp.astype(np.float64) ** 2).sum(), rel=1e-12)
    assert I.min() >= 0


def test_V4_flat_wavefront_symmetries(pyr):
    N, Np, s, bp = 16, 64, 16, 2
    amp = _disc(N, 0.25)
    yx = pyr.valid_pixels(amp, bp)
    sig, Q = pyr.measure(np.zeros((1, N, N), np.float32), amp, yx, Np, s, bp, 3.0, 8, N, return_quadrants=True)
    Sp = N // bp
    grid = np.full((Sp, Sp, 2), np.nan); grid[yx[:, 0], yx[:, 1]] = sig[0]
    # mirror x -> -x maps face b to -b: s_x is antisymmetric in X, s_y symmetric; the same for y
    np.testing.assert_allclose(grid[:, ::-1, 0], -grid[:, :, 0], atol=1e-12, equal_nan=True)
    np.testing.assert_allclose(grid[:, ::-1, 1], grid[:, :, 1], atol=1e-12, equal_nan=True)
    np.testing.assert_allclose(grid[::-1, :, 1], -grid[:, :, 1], atol=1e-12, equal_nan=True)
    assert abs(sig[0, :, 0].sum()) < 1e-12 and abs(sig[0, :, 1].sum()) < 1e-12
    # the four faces carry the same light
    tot = Q[0].sum(axis=(2, 3))
    np.testing.assert_allclose(tot, tot[0, 0], rtol=1e-12)


@pytest.mark.parametrize("tilt", [0.5, 1.0, -1.5])
def test_V5_tilt_response_follows_the_modulated_pyramid_law(pyr, tilt):
    """A tilt of `tilt` lambda/D along x under a circular modulation of radius r_mod: the spot spends the
    fraction asin(tilt/r_mod)/pi more of the cycle on the +x faces: mean s_x = (2/pi) asin(tilt/r_mod)
    (geometric optics; diffraction by a 32-pixel pupil changes it by a few percent), s_y = 0."""
    N, Np, s, bp, r_mod, K = 32, 128, 32, 2, 4.0, 32
    amp = _disc(N)
    yx = pyr.valid_pixels(amp, bp)
    x = np.arange(N, dtype=np.float64)
    ph = np.broadcast_to(2 * np.pi * tilt * x[None, :] / N, (N, N)).astype(np.float32)   # phase grows with x
    sig = pyr.measure(ph[None], amp, yx, Np, s, bp, r_mod, K, N)[0]
    want = (2 / np.pi) * np.arcsin(tilt / r_mod)
    assert sig[:, 0].mean() == pytest.approx(want, rel=0.12)
    assert np.sign(sig[:, 0].mean()) == np.sign(tilt)
    assert abs(sig[:, 1].mean()) < 5e-3
    # along y
    sig_y = pyr.measure(np.ascontiguousarray(ph.T)[None], amp, yx, Np, s, bp, r_mod, K, N)[0]
    assert sig_y[:, 1].mean() == pytest.approx(want, rel=0.12)
    assert abs(sig_y[:, 0].mean()) < 5e-3


def test_V6_transposition_swaps_the_axes(pyr):
    N, Np, s, bp = 16, 64, 16, 2
    amp = _disc(N, 0.2) * rng.uniform(0.6, 1.0, (N, N)).astype(np.float32)
    ampT = np.ascontiguousarray(amp.T)
    ph = rng.normal(0, 1, (N, N)).astype(np.float32)
    yx = pyr.valid_pixels(amp, bp)
    yxT = pyr.valid_pixels(ampT, bp)
    a = pyr.measure(ph[None], amp, yx, Np, s, bp, 2.0, 8, N)[0]
    b = pyr.measure(np.ascontiguousarray(ph.T)[None], ampT, yxT, Np, s, bp, 2.0, 8, N)[0]
    Sp = N // bp
    ga = np.zeros((Sp, Sp, 2)); ga[yx[:, 0], yx[:, 1]] = a
    gb = np.zeros((Sp, Sp, 2)); gb[yxT[:, 0], yxT[:, 1]] = b
    np.testing.assert_allclose(gb[:, :, 0], ga[:, :, 1].T, atol=1e-12)
    np.testing.assert_allclose(gb[:, :, 1], ga[:, :, 0].T, atol=1e-12)


def test_V7_modulation_is_the_average_over_explicit_tilts(pyr):
    """Q1 + Q5: the modulated intensity equals the mean of K unmodulated ones whose wavefront carries the
    modulation tilt r_mod lambda/D towards th_k = 2 pi (k + 1/2) / K, built here in float64."""
    N, Np, s, K, r_mod, D = 16, 64, 16, 4, 2.5, 14.0
    amp = _disc(N, 0.3)
    ph = rng.normal(0, 1, (N, N))
    y, x = np.mgrid[0:N, 0:N].astype(np.float64)
    acc = np.zeros((Np, Np))
    for k in range(K):
        th = 2 * np.pi * (k + 0.5) / K
        acc += pyr.detector_intensity(ph + 2 * np.pi * r_mod * (x * np.cos(th) + y * np.sin(th)) / D, amp, Np, s,
                                      0.0, 0, D)
    np.testing.assert_allclose(pyr.detector_intensity(ph, amp, Np, s, r_mod, K, D), acc / K, atol=1e-13)


def test_V8_piston_is_invisible(pyr):
    N, Np, s, bp = 16, 64, 16, 4
    amp = _disc(N)
    ph = rng.normal(0, 1, (N, N)).astype(np.float32)
    yx = pyr.valid_pixels(amp, bp)
    a = pyr.measure(ph[None], amp, yx, Np, s, bp, 1.0, 4, N)[0]
    b = pyr.measure((ph + np.float32(1.25))[None], amp, yx, Np, s, bp, 1.0, 4, N)[0]
    np.testing.assert_allclose(a, b, atol=1e-6)


def test_V9_each_face_carries_one_focal_plane_quadrant(pyr):
    """The light found around the copy at (+s,+s) is the energy of the focal-plane quadrant u~, v~ > 0 (the
    axes u~ = 0 and the Nyquist line shared half and half): Parseval per face, up to the diffraction tails
    that cross into the neighbouring quarter of the grid (1 %)."""
    N, Np, s = 8, 64, 16
    amp = _disc(N)
    k = np.arange(Np)
    us = np.where(k < Np // 2, k, k - Np)
    w = np.where(us > 0, 1.0, 0.0) + np.where(us == 0, 0.5, 0.0) + np.where(us == -Np // 2, 0.5, 0.0)
    for sd in (1.0, 3.0):
        ph = rng.normal(0, sd, (N, N)).astype(np.float32)
        I = pyr.detector_intensity(ph, amp, Np, s, 0.0, 0, N)
        F = np.fft.fft2(pyr.field(ph, amp, Np, 0.0, 0.0, N))
        want = (np.abs(F) ** 2 * w[None, :] * w[:, None]).sum() / Np ** 2
        assert I[: Np // 2, : Np // 2].sum() == pytest.approx(want, rel=0.01)
        wm = w[::-1].copy(); wm = np.roll(wm, 1)                 # weights of the u~ < 0 half
        want_mm = (np.abs(F) ** 2 * wm[None, :] * wm[:, None]).sum() / Np ** 2
        assert I[Np // 2:, Np // 2:].sum() == pytest.approx(want_mm, rel=0.01)

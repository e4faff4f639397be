"""Pins of the Poisson detector-noise oracle (oracle/shwfs_oracle_poisson.c, steps N1..N5; SURVEY.md 8(f) f2,
PAPER.md:91 "the centroid computed on the final noise-added image").  The paper fixes nothing about the noise, so
the pins are what mathematics fixes about a Poisson draw: the quantile function (a library routine the oracle does
not call), the pmf, the first two moments, the Gaussian limit, independence between counters.  -m "not gpu"."""
import numpy as np
import pytest
from scipy import stats

from oracle import shwfs_oracle as O

SEED = 0x1408_0698


def _draws(lam, n, t=0):
    """n independent draws at rate lam: pixels p of spots i of frame t"""
    ks = np.empty(n, dtype=np.int64)
    ms = np.empty(n)
    for q in range(n):
        ks[q], ms[q] = O.poisson_draw(lam, SEED, t, q // 256, q % 256)
    return ks, ms


def test_P1_inversion_is_the_poisson_quantile_function():
    """N3 returns the smallest k with CDF(k) >= u1: scipy.stats.poisson.ppf, for every u1 clear of a CDF step."""
    rng = np.random.default_rng(1)
    for lam in (0.01, 0.3, 1.0, 3.0, 9.7, 29.9):
        us = np.concatenate([rng.uniform(0, 1, 400), [1e-7, 0.5, 1 - 2.0 ** -24]])
        for u in us:
            k, m = O.poisson_inversion(lam, u)
            if m > 1e-9:
                assert k == int(stats.poisson.ppf(u, lam)), (lam, u, k)
            # the margin is the distance of u to the nearest CDF value the search compared it with
            cdf = stats.poisson.cdf(np.arange(0, k + 1), lam)
            assert m == pytest.approx(np.abs(u - cdf).min(), abs=1e-12)


@pytest.mark.parametrize("lam,n", [(0.3, 40000), (3.0, 40000), (29.9, 20000), (30.0, 20000), (300.0, 20000)])
def test_P2_moments_and_pmf(lam, n):
    """mean = variance = lambda; chi^2 of the histogram against the Poisson pmf (both branches: N3 below 30,
    the transformed rejection N4 from 30 up)."""
    ks, _ = _draws(lam, n)
    assert ks.min() >= 0
    se_mean = np.sqrt(lam / n)
    assert abs(ks.mean() - lam) < 4.5 * se_mean
    se_var = np.sqrt((lam + 2 * lam * lam) / n)            # var of the sample variance of a Poisson variable, ~
    assert abs(ks.var(ddof=1) - lam) < 4.5 * se_var
    lo, hi = int(stats.poisson.ppf(1e-3, lam)), int(stats.poisson.ppf(1 - 1e-3, lam))
    edges = np.arange(lo, hi + 2)
    obs = np.histogram(np.clip(ks, lo, hi), bins=edges)[0].astype(float)
    p = stats.poisson.pmf(np.arange(lo, hi + 1), lam)
    p[0] = stats.poisson.cdf(lo, lam)
    p[-1] = stats.poisson.sf(hi - 1, lam)
    # merge cells with an expectation below 5
    exp = n * p
    keep = exp >= 5
    obs_m = np.append(obs[keep], obs[~keep].sum())
    exp_m = np.append(exp[keep], exp[~keep].sum())
    if exp_m[-1] < 5:
        obs_m[-2] += obs_m[-1]; exp_m[-2] += exp_m[-1]
        obs_m, exp_m = obs_m[:-1], exp_m[:-1]
    chi2 = ((obs_m - exp_m) ** 2 / exp_m).sum()
    assert stats.chi2.sf(chi2, len(exp_m) - 1) > 1e-4, (lam, chi2, len(exp_m))


def test_P3_gaussian_limit():
    """lambda = 1e4: (k - lambda) / sqrt(lambda) is N(0,1) to the skewness 1/sqrt(lambda) -- the limit in which
    reading B4 (photon_model 0) and the Poisson model agree."""
    lam = 1.0e4
    ks, _ = _draws(lam, 8000)
    zz = (ks - lam) / np.sqrt(lam)
    assert stats.kstest(zz, "norm").pvalue > 1e-3
    assert abs(zz.mean()) < 0.05 and abs(zz.std() - 1) < 0.04


def test_P4_degenerate_rates():
    assert O.poisson_draw(0.0, SEED, 0, 0, 0) == (0, 1.0)
    B = np.zeros((4, 4)); B[1, 2] = -3.0                      # a negative rate is clipped (N1)
    c = O.add_noise_poisson(B, 5.0, 0.0, SEED, 0, 0)
    assert np.all(c == 0.0)
    np.testing.assert_array_equal(O.add_noise_poisson(B, 0.0, 2.0, SEED, 0, 0), B)     # F <= 0: no noise


def test_P5_counter_layout_and_independence():
    """N2: pixel p takes words (2 (p mod 2), +1) of the block with counter (p/2, i, t, 1 + j); different pixels,
    spots, frames and attempts see different uniforms; the draws of neighbouring pixels are uncorrelated."""
    key = np.array([SEED & 0xFFFFFFFF, SEED >> 32], dtype=np.uint32)
    for (t, i, p, j) in ((0, 0, 0, 0), (3, 17, 5, 0), (3, 17, 4, 2), (1000, 4631, 255, 7)):
        x = O.philox4x32(np.array([p // 2, i, t, 1 + j], dtype=np.uint32), key)
        w = 2 * (p % 2)
        want = ((x[w:w + 2] >> 9).astype(np.float64) + 0.5) / 8388608.0
        np.testing.assert_array_equal(O.poisson_uniforms(SEED, t, i, p, j), want)
    seen = {tuple(O.poisson_uniforms(SEED, t, i, p, j)) for t in range(3) for i in range(3) for p in range(6)
            for j in range(2)}
    assert len(seen) == 3 * 3 * 6 * 2
    B = np.full((16, 16), 4.0)
    imgs = np.stack([O.add_noise_poisson(B, 1.0, 0.0, SEED, t, 0) for t in range(300)])     # [300,16,16]
    flat = imgs.reshape(300, -1) - 4.0
    cc = np.corrcoef(flat.T)
    off = cc[~np.eye(256, dtype=bool)]
    assert abs(off.mean()) < 0.01 and np.abs(off).max() < 0.35        # 300 samples: |r| ~ 0.06 rms


def test_P6_read_noise_term():
    """N5: counts = k + ron z with z the deviate of L5 (block p/4, deviate p mod 4): subtracting the Poisson part
    leaves exactly ron z, and the variance is lambda + ron^2."""
    B = np.random.default_rng(5).uniform(0.5, 6.0, (16, 16))
    F, ron, t, i = 2.0, 3.0, 4, 9
    c0 = O.add_noise_poisson(B, F, 0.0, SEED, t, i)
    c3 = O.add_noise_poisson(B, F, ron, SEED, t, i)
    z = np.empty((16, 16))
    for Cc in range(16):
        for R in range(16):
            p = Cc * 16 + R
            z[R, Cc] = O.normal4(SEED, t, i, p // 4)[p % 4]
    np.testing.assert_allclose(c3 - c0, ron * z, rtol=0, atol=1e-12)
    assert np.all(c0 == np.round(c0))
    Bc = np.full((16, 16), 5.0)
    v = np.stack([O.add_noise_poisson(Bc, 1.0, 2.0, SEED, tt, 0) for tt in range(200)]).ravel()
    assert abs(v.mean() - 5.0) < 0.06 and abs(v.var() - 9.0) < 0.35


def test_P7_measure_lgs_threads_the_model_through():
    """photon_model = 1 of the whole-call routine is N1..N5 applied to its own binned image (stage 2 -> stage 3)."""
    from paper_1408_0698_b200 import workloads as W
    c = W.CONFIGS[1]
    amp = W.pupil_mask(c)
    yx = O.valid_list(amp, c.n, c.min_illum)[:6]
    ph = W.phase_frames(c, 0, range(2))
    kw = dict(weight=[1.0], defocus=[0.0], tau=0.1, flux=3.0, ron=1.5, seed=SEED)
    _, b2 = O.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, stage=2, photon_model=1, **kw)
    s3, b3, mg = O.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, stage=3, photon_model=1, want_margins=True, **kw)
    for t in range(2):
        for i in range(len(yx)):
            want, m = O.add_noise_poisson(b2[t, i], 3.0, 1.5, SEED, t, i, want_margin=True)
            np.testing.assert_array_equal(b3[t, i], want)
            np.testing.assert_array_equal(mg[t, i], m)
            np.testing.assert_allclose(s3[t, i], O.threshold_cog(b3[t, i], 0.1, 0), atol=1e-12)
    # photon_model 0 is untouched
    _, g3 = O.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, stage=3, **kw)
    np.testing.assert_allclose(g3[0, 0], O.add_noise(b2[0, 0], 3.0, 1.5, SEED, 0, 0), atol=1e-12)

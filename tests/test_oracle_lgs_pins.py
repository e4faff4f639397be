"""Pins of the float64 oracle of the paper's full LGS model (oracle/shwfs_oracle_lgs.c): sodium sub-layer
sum and detector noise (f2).

As in test_oracle_pins.py nothing here compares a function with itself: J1 reduces to the already pinned
single-layer routine, J2 is brute-force linearity, J3-J5 are closed forms / symmetries, J6 the generator's
published known-answer vectors (tests/golden/philox4x32_10_kat.txt), J7-J9 distribution facts.  CPU only.
"""
from pathlib import Path

import numpy as np
import pytest

rng = np.random.default_rng(91)
SIZES = [(8, 16, 1), (10, 32, 2), (16, 64, 4)]


def _pupil(n, S=4, partial=True):
    N = n * S
    amp = np.ones((N, N), np.float32)
    if partial:
        amp[: n // 2, : n // 3] = 0.0
        amp[N - 2:, N - n:] = 0.5
    yx = np.array([[sy, sx] for sy in range(S) for sx in range(S)], np.int32)
    return amp, yx, N


def _kern(P, nsub, seed=5):
    k = np.random.default_rng(seed).random((nsub, P, P)).astype(np.float32)
    return k / k.sum(axis=(1, 2), keepdims=True)


# ---------------------------------------------------------------- J1
@pytest.mark.parametrize("n,P,b", SIZES)
@pytest.mark.parametrize("elong", [False, True])
def test_J1_one_plain_layer_is_the_single_layer_sensor(oracle, n, P, b, elong):
    amp, yx, N = _pupil(n)
    ph = rng.normal(0, 2.0, (2, N, N)).astype(np.float32)
    K = _kern(P, len(yx)) if elong else None
    want, wimg = oracle.measure(ph, amp, yx, n, P, b, tau=0.1, kernels=K, stage=2, c_phi=0.8)
    for shared in (True, False):
        p = ph if shared else ph[:, None]
        got, img = oracle.measure_lgs(p, amp, yx, n, P, b, 0.05, weight=[1.0], defocus=[0.0], tau=0.1,
                                      kernels=K, stage=2, c_phi=0.8)
        np.testing.assert_allclose(img, wimg, rtol=0, atol=1e-13 * wimg.max())
        np.testing.assert_allclose(got, want, rtol=0, atol=1e-12)


# ---------------------------------------------------------------- J2
@pytest.mark.parametrize("n,P,b", SIZES)
def test_J2_image_is_weighted_sum_of_layer_images(oracle, n, P, b):
    """L2+L3: B = sum_l w_l B_l, each B_l from the single-layer routine on a wavefront that already holds
    that layer's analytic phase (built here in float64 and fed through c_phi = 1 as an fp32 input is not
    exact, so the analytic part is put into the phase of a one-layer call instead)."""
    amp, yx, N = _pupil(n)
    L, dx = 3, 0.05
    ph = rng.normal(0, 1.5, (2, L, N, N)).astype(np.float32)
    w = np.array([0.2, 0.5, 0.3])
    de = np.array([-0.8, 0.1, 0.9])
    tx = np.array([0.3, 0.0, -0.2]) / dx
    ty = np.array([-0.1, 0.2, 0.05]) / dx
    K = _kern(P, len(yx))
    kw = dict(cx=0.12, cy=-0.07, kernels=K, c_phi=1.0)
    got, img = oracle.measure_lgs(ph, amp, yx, n, P, b, dx, weight=w, defocus=de, tilt_x=tx, tilt_y=ty,
                                  stage=2, **kw)
    acc = np.zeros_like(img)
    for l in range(L):
        _, one = oracle.measure_lgs(np.ascontiguousarray(ph[:, l]), amp, yx, n, P, b, dx, weight=[1.0],
                                    defocus=[de[l]], tilt_x=[tx[l]], tilt_y=[ty[l]], stage=2, **kw)
        acc += w[l] * one
    np.testing.assert_allclose(img, acc, rtol=0, atol=1e-12 * acc.max())
    # and the slopes are the centre of gravity of that image (O8/O9, pinned in test_oracle_pins.py)
    for t in range(2):
        for i in range(len(yx)):
            np.testing.assert_allclose(got[t, i], oracle.threshold_cog(img[t, i], 0.0, 0), atol=1e-12)


# ---------------------------------------------------------------- J3
@pytest.mark.parametrize("n,P,b", SIZES)
def test_J3_layer_tilt_of_whole_pixels_shifts_the_spot_exactly(oracle, n, P, b):
    """g = 2*pi*m/(P*dx) rad/m is m unbinned pixels: the layer image is the untilted one rolled by (my,mx)."""
    amp, yx, N = _pupil(n)
    dx = 0.07
    ph = rng.normal(0, 1.0, (1, N, N)).astype(np.float32)
    mx, my = 2 * b, -b                     # whole detector pixels so that the binned images roll too
    base = oracle.measure_lgs(ph, amp, yx, n, P, b, dx, weight=[1.0], defocus=[0.0], stage=2)[1]
    g = 2 * np.pi / (P * dx)
    tilt = oracle.measure_lgs(ph, amp, yx, n, P, b, dx, weight=[1.0], defocus=[0.0], tilt_x=[mx * g],
                              tilt_y=[my * g], stage=2)[1]
    want = np.roll(base, (my // b, mx // b), axis=(2, 3))
    np.testing.assert_allclose(tilt, want, rtol=0, atol=1e-11 * base.max())


# ---------------------------------------------------------------- J4
@pytest.mark.parametrize("n,P,b", SIZES)
def test_J4_defocus_displaces_each_spot_by_its_local_gradient(oracle, n, P, b):
    """A quadratic a|r - r_c|^2 on a flat wavefront is, over subaperture i, a tilt 2a(r_i - r_c) plus a
    symmetric curvature: the centroid moves by 2a(r_i - r_c) dx P / (2 pi b) detector pixels (linear range,
    5 % as in I3).  Catches a missing factor 2, a sign, swapped axes and a wrong pixel-centre convention."""
    amp, yx, N = _pupil(n, partial=False)
    dx = 0.05
    cx, cy = 0.031, -0.042
    ph = np.zeros((1, N, N), np.float32)
    S = N // n
    r_max = (S / 2) * n * dx
    a = 0.25 * (2 * np.pi / P) / (2 * r_max * dx)      # <= 0.25 unbinned px of shift at the pupil edge
    got = oracle.measure_lgs(ph, amp, yx, n, P, b, dx, weight=[1.0], defocus=[a], cx=cx, cy=cy)[0]
    xc = ((yx[:, 1] + 0.5) * n - N / 2) * dx
    yc = ((yx[:, 0] + 0.5) * n - N / 2) * dx
    want_x = 2 * a * (xc - cx) * dx * P / (2 * np.pi * b)
    want_y = 2 * a * (yc - cy) * dx * P / (2 * np.pi * b)
    assert np.abs(want_x).max() > 0.05 / b
    np.testing.assert_allclose(got[:, 0], want_x, rtol=0.05, atol=2e-3)
    np.testing.assert_allclose(got[:, 1], want_y, rtol=0.05, atol=2e-3)
    assert not np.allclose(got[:, 0], got[:, 1], atol=1e-3)


# ---------------------------------------------------------------- J5
@pytest.mark.parametrize("n,P,b", SIZES)
@pytest.mark.parametrize("tau", [0.0, 0.15])
def test_J5_opposite_layers_cancel(oracle, n, P, b, tau):
    """Layers (a, g) and (-a, -g) with equal weights on a flat wavefront: the second spot is the point
    reflection of the first (I8), so the sum is point symmetric and its centre of gravity is zero."""
    amp, yx, N = _pupil(n, partial=False)
    dx = 0.05
    ph = np.full((1, N, N), 0.7, np.float32)
    got = oracle.measure_lgs(ph, amp, yx, n, P, b, dx, weight=[0.5, 0.5], defocus=[1.3, -1.3],
                             tilt_x=[4.0, -4.0], tilt_y=[-2.5, 2.5], cx=0.2, cy=0.1, tau=tau)
    assert np.abs(got).max() < 1e-12
    one = oracle.measure_lgs(ph, amp, yx, n, P, b, dx, weight=[1.0], defocus=[1.3], tilt_x=[4.0],
                             tilt_y=[-2.5], cx=0.2, cy=0.1, tau=tau)
    assert np.abs(one).max() > 1e-2


# ---------------------------------------------------------------- J6
def test_J6_philox4x32_10_known_answers(oracle):
    rows = [l.split() for l in (Path(__file__).parent / "golden" / "philox4x32_10_kat.txt").read_text().splitlines()
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = oracle.philox4x32(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


# ---------------------------------------------------------------- J7
def test_J7_deviates_are_standard_normal_and_uncorrelated(oracle):
    from scipy import stats
    z = np.array([oracle.normal4(12345, t, i, blk) for t in range(8) for i in range(25) for blk in range(64)])
    flat = z.reshape(-1)                                  # 51 200 deviates
    assert abs(flat.mean()) < 4 / np.sqrt(flat.size)
    assert abs(flat.var() - 1) < 4 * np.sqrt(2 / flat.size)
    assert abs(stats.skew(flat)) < 0.05 and abs(stats.kurtosis(flat)) < 0.1
    assert stats.kstest(flat, "norm").pvalue > 1e-3
    c = np.corrcoef(z.T)                                  # the four deviates of a block
    assert np.abs(c - np.eye(4)).max() < 0.03
    zz = z.reshape(8, 25, 64, 4)
    assert abs(np.corrcoef(zz[0].reshape(-1), zz[1].reshape(-1))[0, 1]) < 0.03      # frames
    assert abs(np.corrcoef(zz[:, 0].reshape(-1), zz[:, 1].reshape(-1))[0, 1]) < 0.03  # subapertures
    assert abs(np.corrcoef(zz[:, :, :-1].reshape(-1), zz[:, :, 1:].reshape(-1))[0, 1]) < 0.02  # blocks
    assert not np.allclose(oracle.normal4(12345, 0, 0, 0), oracle.normal4(12346, 0, 0, 0))


# ---------------------------------------------------------------- J8
def test_J8_counts_have_mean_FB_and_variance_FB_plus_ron2(oracle):
    D = 16
    B = np.random.default_rng(2).random((D, D)) * 3.0
    B[0, 0] = 0.0
    B[3, 4] = -1e-9                                       # rounding-level negative: variance uses max(.,0)
    F, ron = 40.0, 3.0
    c = np.array([oracle.add_noise(B, F, ron, 77, t, 5) for t in range(4000)])
    m, v = c.mean(axis=0), c.var(axis=0)
    want_v = np.maximum(F * B, 0) + ron ** 2
    assert np.abs(m - F * B).max() < 5 * np.sqrt(want_v.max() / 4000)
    np.testing.assert_allclose(v, want_v, rtol=0.12)
    assert np.isfinite(c).all()
    # pixel p = C*D + R takes deviate p % 4 of block p / 4 (column-major)
    one = oracle.add_noise(B, F, ron, 77, 0, 5)
    R, C = 6, 9
    z = oracle.normal4(77, 0, 5, (C * D + R) // 4)[(C * D + R) % 4]
    assert one[R, C] == pytest.approx(F * B[R, C] + np.sqrt(F * B[R, C] + ron ** 2) * z, abs=1e-12)
    np.testing.assert_array_equal(oracle.add_noise(B, 0.0, ron, 77, 0, 5), B)


# ---------------------------------------------------------------- J9
def test_J9_large_flux_recovers_noise_free_slopes(oracle):
    n, P, b = 10, 32, 2
    amp, yx, N = _pupil(n)
    ph = rng.normal(0, 1.0, (2, N, N)).astype(np.float32)
    kw = dict(weight=[0.6, 0.4], defocus=[0.5, -0.4], tau=0.1, kernels=_kern(P, len(yx)))
    clean = oracle.measure_lgs(ph, amp, yx, n, P, b, 0.05, **kw)
    err = []
    for F in (1e2, 1e4, 1e6):
        noisy = oracle.measure_lgs(ph, amp, yx, n, P, b, 0.05, flux=F, ron=0.0, seed=3, **kw)
        err.append(np.abs(noisy - clean).max())
    assert err[0] > err[1] > err[2] and err[2] < 2e-2 and err[0] > 1e-2
    ratio = err[0] / err[2]
    assert 30 < ratio < 300                               # photon noise scales as 1/sqrt(F): 100 expected
    # stage 3 is stage 2 plus the L4 noise of the same (seed, t, i)
    _, b2 = oracle.measure_lgs(ph, amp, yx, n, P, b, 0.05, flux=50.0, ron=2.0, seed=9, stage=2, **kw)
    _, b3 = oracle.measure_lgs(ph, amp, yx, n, P, b, 0.05, flux=50.0, ron=2.0, seed=9, stage=3, **kw)
    np.testing.assert_allclose(b3[1, 7], oracle.add_noise(b2[1, 7], 50.0, 2.0, 9, 1, 7), atol=1e-12)

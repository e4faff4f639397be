"""Pins of the closed-loop oracle (oracle/closed_loop.py).  CPU only."""
import numpy as np
import pytest

rng = np.random.default_rng(76)


def _setup(n=8, P=16, b=1, S=4):
    N = n * S
    amp = np.ones((N, N), np.float32)
    yx = np.array([[sy, sx] for sy in range(S) for sx in range(S)], np.int32)
    ax = (np.arange(N) + 0.5 - N / 2)
    tilt_x = np.broadcast_to(ax[None, :], (N, N)).copy()
    tilt_y = np.broadcast_to(ax[:, None], (N, N)).copy()
    return N, amp, yx, np.stack([tilt_x, tilt_y]) * (2 * np.pi / P)      # 1 unit = 1 unbinned px of shift


@pytest.fixture(scope="module")
def loop():
    from oracle import closed_loop
    return closed_loop


def test_K1_zero_coefficients_leave_the_wavefront(loop):
    ph = rng.normal(0, 1, (3, 12, 12)).astype(np.float32)
    modes = rng.normal(0, 1, (5, 12, 12))
    res = loop.residual_phase(ph, modes, np.zeros((3, 5)))
    np.testing.assert_array_equal(res, ph.astype(np.float64))


def test_K2_a_mode_combination_is_cancelled(loop, oracle):
    n, P, b = 8, 16, 1
    N, amp, yx, _ = _setup(n, P, b)
    modes = rng.normal(0, 1, (6, N, N))
    c = rng.normal(0, 1, (2, 6))
    ph = np.einsum("tm,myx->tyx", c, modes)
    res = loop.residual_phase(ph, modes, c)
    assert np.abs(res).max() < 1e-13
    s = loop.measure_residual(ph, modes, c, amp, yx, n, P, b, tau=0.1)
    assert np.abs(s).max() < 1e-6                      # fp32 rounding of a ~1e-15 residual: flat wavefront


def test_K3_einsum_restatement_and_slope_order(loop):
    ph = rng.normal(0, 1, (4, 10, 10)).astype(np.float32)
    modes = rng.normal(0, 1, (7, 10, 10))
    c = rng.normal(0, 1, (4, 7))
    np.testing.assert_allclose(loop.residual_phase(ph, modes, c),
                               ph - np.einsum("tm,myx->tyx", c, modes), atol=1e-13)
    nsub, M = 9, 5
    R = rng.normal(0, 1, (M, 2 * nsub))
    s = rng.normal(0, 1, (3, nsub, 2))
    want = np.einsum("mia,tia->tm", R.reshape(M, nsub, 2), s)       # k = 2*i + axis
    np.testing.assert_allclose(loop.reconstruct(R, s), want, atol=1e-13)
    # a matrix that picks the y-slope of subaperture 4
    pick = np.zeros((1, 2 * nsub)); pick[0, 2 * 4 + 1] = 1.0
    np.testing.assert_allclose(loop.reconstruct(pick, s)[:, 0], s[:, 4, 1])


@pytest.mark.parametrize("gain", [0.3, 0.6, 1.0])
def test_K4_static_tilt_converges_as_one_minus_gain_to_the_t(loop, gain):
    """Pure integrator on a static aberration a: c_t = a (1 - (1-g)^t), so the residual coefficient is
    a (1-g)^t (sensor in its linear range: 0.06 px tilts, plain CoG)."""
    n, P, b = 8, 16, 1
    N, amp, yx, modes = _setup(n, P, b)
    D = loop.interaction_matrix(modes, amp, yx, n, P, b)
    R = np.linalg.pinv(D)
    a = np.array([0.06, -0.045])                                # near the calibration amplitude: linear
    T = 7
    ph = np.broadcast_to(np.einsum("m,myx->yx", a, modes), (T, N, N)).astype(np.float32)
    slopes, hist, cT = loop.closed_loop(ph, modes, R, gain, np.zeros(2), amp, yx, n, P, b)
    want = a[None, :] * (1 - (1 - gain) ** np.arange(T))[:, None]
    np.testing.assert_allclose(hist, want, atol=5e-4)
    np.testing.assert_allclose(cT, a * (1 - (1 - gain) ** T), atol=5e-4)
    assert hist[0].tolist() == [0.0, 0.0]                       # C4: hist[t] is what shaped frame t
    # C3 delay: the slopes of frame 0 see the full aberration, those of frame t the residual a (1-g)^t
    sx = slopes[:, :, 0].mean(axis=1)
    assert abs(sx[0] / a[0] - 1.0) < 0.05                       # sensor gain ~ 1/b (I3), not exactly 1
    np.testing.assert_allclose(sx / sx[0], (1 - gain) ** np.arange(T), atol=4e-3)


def test_K5_zero_gain_freezes_wrong_sign_diverges(loop):
    n, P, b = 8, 16, 1
    N, amp, yx, modes = _setup(n, P, b)
    R = np.linalg.pinv(loop.interaction_matrix(modes, amp, yx, n, P, b))
    a = np.array([0.2, 0.1])
    ph = np.broadcast_to(np.einsum("m,myx->yx", a, modes), (5, N, N)).astype(np.float32)
    _, hist, cT = loop.closed_loop(ph, modes, R, 0.0, np.array([0.05, 0.0]), amp, yx, n, P, b)
    assert (hist == np.array([0.05, 0.0])).all() and (cT == np.array([0.05, 0.0])).all()
    _, hist, _ = loop.closed_loop(ph, modes, -R, 0.5, np.zeros(2), amp, yx, n, P, b)
    err = np.abs(a - hist).max(axis=1)
    assert (np.diff(err) > 0).all()                              # runs away from the aberration


def test_interaction_matrix_of_tilts_is_the_tilt_closed_form(loop):
    """PAPER.md:69 push-pull on tilt modes: one unbinned pixel of tilt moves every spot by 1/b detector px
    along that axis and not along the other (I3 of the sensor, seen through the calibration)."""
    n, P, b = 10, 32, 2
    N, amp, yx, modes = _setup(n, P, b)
    D = loop.interaction_matrix(modes, amp, yx, n, P, b, amp_push=0.1)
    Dx = D.reshape(len(yx), 2, 2)
    np.testing.assert_allclose(Dx[:, 0, 0], 1.0 / b, rtol=0.05)
    np.testing.assert_allclose(Dx[:, 1, 1], 1.0 / b, rtol=0.05)
    assert np.abs(Dx[:, 0, 1]).max() < 1e-10 and np.abs(Dx[:, 1, 0]).max() < 1e-10

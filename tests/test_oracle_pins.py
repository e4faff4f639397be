"""Pins of the float64 oracle against what the mathematics fixes.

None of these compares the oracle with itself: each checks a closed form, an invariant, a brute-force
definition or a library routine (numpy.fft) that a plausible mistake in oracle/shwfs_oracle.c -- a dropped
term, a wrong sign or index, a transposed operand -- would break.  CPU only.
"""
import numpy as np
import pytest

from paper_1408_0698_b200 import workloads as W

SIZES = [(8, 16, 1), (16, 32, 2), (10, 32, 2), (16, 64, 4)]      # (n, P, b) of configs 1, 2, 3-4, 5
rng = np.random.default_rng(1408)


def _one_sub(n, mask=None):
    """A pupil of exactly one subaperture: N = n, valid list [(0,0)]."""
    amp = np.ones((n, n), np.float32) if mask is None else mask.astype(np.float32)
    return amp, np.array([[0, 0]], np.int32)


def _partial_mask(n):
    m = np.ones((n, n), np.float32)
    m[: n // 3, : n // 2] = 0.0          # asymmetric, ~17 % dark
    m[n - 1, n - 2:] = 0.0
    return m


def _sym_kernel(P, seed=3):
    """Random positive kernel, point-symmetric about (P/2, P/2) on the periodic grid, sum 1."""
    k = np.random.default_rng(seed).random((P, P))
    idx = (P - np.arange(P)) % P
    kc = np.roll(k, (-P // 2, -P // 2), (0, 1))         # centre to the origin
    kc = 0.5 * (kc + kc[np.ix_(idx, idx)])
    k = np.roll(kc, (P // 2, P // 2), (0, 1))
    return (k / k.sum()).astype(np.float32)


# ---------------------------------------------------------------- I1
@pytest.mark.parametrize("n,P,b", SIZES)
@pytest.mark.parametrize("tau", [0.0, 0.1])
@pytest.mark.parametrize("elong", [False, True])
@pytest.mark.parametrize("partial", [False, True])
def test_I1_flat_wavefront_gives_zero_slopes(oracle, n, P, b, tau, elong, partial):
    amp, yx = _one_sub(n, _partial_mask(n) if partial else None)
    K = _sym_kernel(P)[None] if elong else None
    for piston in (0.0, 1.2345):
        ph = np.full((1, n, n), piston, np.float32)
        s = oracle.measure(ph, amp, yx, n, P, b, tau=tau, kernels=K)
        assert np.abs(s).max() < 1e-13


# ---------------------------------------------------------------- I2
@pytest.mark.parametrize("n,P,b", SIZES)
def test_I2_integer_tilt_is_exact_circular_shift(oracle, n, P, b):
    amp, yx = _one_sub(n, _partial_mask(n))
    ph = rng.normal(0, 1.0, (1, n, n)).astype(np.float32)
    j, k = np.mgrid[0:n, 0:n]
    mx, my = 3, -2
    # the tilt is applied in float64 through c_phi = 1 on an fp32 input, so build it as an exact
    # separate frame: use phase_to_rad to keep the fp32 rounding of the sum out of the comparison
    tilt = 2 * np.pi * (mx * k + my * j) / P
    _, i0 = oracle.measure(ph, amp, yx, n, P, b, stage=0)
    ph64 = ph[0].astype(np.float64) + tilt
    ph_t = ph64.astype(np.float32)[None]
    _, i1 = oracle.measure(ph_t, amp, yx, n, P, b, stage=0)
    want = np.roll(i0[0, 0], (my, mx), (0, 1))
    # fp32 rounding of the tilted input (|phase| <~ 10 rad -> 5e-7 rad) bounds the error
    assert np.abs(i1[0, 0] - want).max() < 2e-5 * want.max()
    # x is the fast axis: a pure x-tilt of the flat spot moves its 2x2 peak block by +mx COLUMNS only
    ones = np.ones((n, n), np.float32)
    _, f1 = oracle.measure((2 * np.pi * mx * k / P).astype(np.float32)[None], ones, yx, n, P, b, stage=0)
    r, c = np.unravel_index(np.argmax(f1[0, 0]), (P, P))
    assert r in (P // 2 - 1, P // 2) and c in (P // 2 - 1 + mx, P // 2 + mx)


def test_I2_slopes_change_by_m_over_b(oracle):
    n, P, b = 10, 32, 2
    amp, yx = _one_sub(n)
    j, k = np.mgrid[0:n, 0:n]
    ph = (0.3 * np.sin(0.7 * k) * np.cos(0.4 * j)).astype(np.float64)
    s0 = oracle.measure(ph.astype(np.float32)[None], amp, yx, n, P, b, tau=0.1)
    ph2 = ph + 2 * np.pi * (2 * k - 4 * j) / P
    s1 = oracle.measure(ph2.astype(np.float32)[None], amp, yx, n, P, b, tau=0.1)
    assert np.allclose(s1 - s0, [[[2 / b, -4 / b]]], atol=2e-5)


# ---------------------------------------------------------------- I3
@pytest.mark.parametrize("n,P,b", SIZES)
@pytest.mark.parametrize("s_px", [-0.25, 0.1, 0.2])
def test_I3_small_tilt_closed_form(oracle, n, P, b, s_px):
    """Tilt of s unbinned pixels (phase 2*pi*s*k/P) displaces the spot by s/b detector px (tau=0, 5 %)."""
    amp, yx = _one_sub(n)
    j, k = np.mgrid[0:n, 0:n]
    sx = oracle.measure((2 * np.pi * s_px * k / P).astype(np.float32)[None], amp, yx, n, P, b)[0, 0]
    sy = oracle.measure((2 * np.pi * s_px * j / P).astype(np.float32)[None], amp, yx, n, P, b)[0, 0]
    assert abs(sx[0] - s_px / b) < 0.05 * abs(s_px / b) and abs(sx[1]) < 1e-7
    assert abs(sy[1] - s_px / b) < 0.05 * abs(s_px / b) and abs(sy[0]) < 1e-7
    assert np.sign(sx[0]) == np.sign(s_px)        # positive slope <=> phase increasing with x (A4)


def test_I3_half_pixel_tilt_is_exact(oracle):
    n, P, b = 10, 32, 1
    amp, yx = _one_sub(n)
    j, k = np.mgrid[0:n, 0:n]
    s = oracle.measure((2 * np.pi * 0.5 * k / P).astype(np.float32)[None], amp, yx, n, P, b)[0, 0]
    assert abs(s[0] - 0.5) < 1e-6 and abs(s[1]) < 1e-6


# ---------------------------------------------------------------- I4
@pytest.mark.parametrize("n,P,b", SIZES)
def test_I4_parseval_and_flux_conservation(oracle, n, P, b):
    amp = _partial_mask(n) * rng.uniform(0.5, 1.0, (n, n)).astype(np.float32)
    yx = np.array([[0, 0]], np.int32)
    ph = rng.normal(0, 2.0, (1, n, n)).astype(np.float32)
    K = (rng.random((1, P, P)) * 0.01).astype(np.float32)             # not normalised on purpose
    _, I = oracle.measure(ph, amp, yx, n, P, b, stage=0)
    _, Sh = oracle.measure(ph, amp, yx, n, P, b, kernels=K, stage=1)
    _, B = oracle.measure(ph, amp, yx, n, P, b, kernels=K, stage=2)
    flux = float((amp.astype(np.float64) ** 2).sum())
    assert abs(I.sum() - flux) < 1e-12 * flux
    assert abs(Sh.sum() - flux * K.astype(np.float64).sum()) < 1e-12 * flux
    assert abs(B.sum() - Sh.sum()) < 1e-12 * flux


# ---------------------------------------------------------------- I5
@pytest.mark.parametrize("P", [4, 8, 16, 32])
def test_I5_fft_equals_bruteforce_dft(oracle, P):
    x = rng.normal(size=(P, P)) + 1j * rng.normal(size=(P, P))
    for sign in (-1, +1):
        assert np.abs(oracle.dft2(x, sign) - oracle.dft2_brute(x, sign)).max() < 1e-11


@pytest.mark.parametrize("P", [16, 32, 64])
def test_I5_dft_sign_axes_and_library(oracle, P):
    x = rng.normal(size=(P, P)) + 1j * rng.normal(size=(P, P))
    assert np.abs(oracle.dft2(x, -1) - np.fft.fft2(x)).max() < 1e-10
    assert np.abs(oracle.dft2(x, +1) - np.fft.ifft2(x) * P * P).max() < 1e-10
    d = np.zeros((P, P), complex)
    d[1, 0] = 1.0                           # delta at row 1 -> exp(-2 pi i v / P) along rows v
    got = oracle.dft2(d, -1)
    want = np.exp(-2j * np.pi * np.arange(P) / P)[:, None] * np.ones((1, P))
    assert np.abs(got - want).max() < 1e-12


# ---------------------------------------------------------------- I6
@pytest.mark.parametrize("n,P,b", SIZES)
def test_I6_point_symmetric_phase_gives_symmetric_spot(oracle, n, P, b):
    amp, yx = _one_sub(n)
    q = rng.normal(0, 1.5, (n, n))
    ph = (0.5 * (q + q[::-1, ::-1])).astype(np.float32)[None]
    s, Sh = oracle.measure(ph, amp, yx, n, P, b, kernels=_sym_kernel(P)[None], tau=0.1, stage=1)
    assert np.abs(Sh[0, 0] - Sh[0, 0][::-1, ::-1]).max() < 1e-13 * Sh.max()
    assert np.abs(s).max() < 1e-12


# ---------------------------------------------------------------- I7
def test_I7_piston_and_2pi_invariance(oracle):
    n, P, b = 10, 32, 2
    amp, yx = _one_sub(n, _partial_mask(n))
    ph = rng.normal(0, 2.0, (n, n))
    base = oracle.measure(ph.astype(np.float32)[None], amp, yx, n, P, b, tau=0.1)
    wrap = 2 * np.pi * rng.integers(-3, 4, (n, n))
    for other in (ph + 0.777, ph + wrap):
        s = oracle.measure(other.astype(np.float32)[None], amp, yx, n, P, b, tau=0.1)
        assert np.abs(s - base).max() < 2e-5          # fp32 rounding of the shifted input only


# ---------------------------------------------------------------- I8
@pytest.mark.parametrize("n,P,b", SIZES)
def test_I8_phase_negation_reflects_the_spot(oracle, n, P, b):
    amp, yx = _one_sub(n, _partial_mask(n))
    ph = rng.normal(0, 1.5, (1, n, n)).astype(np.float32)
    K = _sym_kernel(P)[None]
    sp, ip = oracle.measure(ph, amp, yx, n, P, b, kernels=K, tau=0.1, stage=1)
    sm, im = oracle.measure(-ph, amp, yx, n, P, b, kernels=K, tau=0.1, stage=1)
    assert np.abs(im[0, 0] - ip[0, 0][::-1, ::-1]).max() < 1e-13 * ip.max()
    assert np.abs(sm + sp).max() < 1e-12 and np.abs(sp).max() > 1e-3


# ---------------------------------------------------------------- I9
@pytest.mark.parametrize("n,P,b", SIZES)
def test_I9_transpose_swaps_x_and_y(oracle, n, P, b):
    amp, yx = _one_sub(n, _partial_mask(n))
    ph = rng.normal(0, 1.5, (n, n)).astype(np.float32)
    s = oracle.measure(ph[None], amp, yx, n, P, b, tau=0.1)[0, 0]
    st = oracle.measure(ph.T.copy()[None], amp.T.copy(), yx, n, P, b, tau=0.1)[0, 0]
    assert np.abs(st - s[::-1]).max() < 1e-13 and abs(s[0] - s[1]) > 1e-3


# ---------------------------------------------------------------- I10, I14, I15
def test_I10_threshold_is_relative(oracle):
    B = rng.random((16, 16))
    for mode in (0, 1):
        a = oracle.threshold_cog(B, 0.1, mode)
        c = oracle.threshold_cog(B * 37.5, 0.1, mode)
        assert np.abs(a - c).max() < 1e-13


def test_I14_single_lit_pixel(oracle):
    D = 16
    for (R, Cc) in [(0, 0), (3, 11), (15, 2)]:
        B = np.zeros((D, D))
        B[R, Cc] = 2.5
        for tau in (0.0, 0.1):
            s = oracle.threshold_cog(B, tau, 0)
            assert np.allclose(s, [Cc - (D - 1) / 2, R - (D - 1) / 2], atol=1e-14)
    assert np.all(oracle.threshold_cog(np.zeros((D, D)), 0.1, 0) == 0.0)


def test_O8_threshold_semantics_by_hand(oracle):
    B = np.array([[10.0, 2.0], [0.5, 4.0]])                 # D = 2, reference (D-1)/2 = 0.5
    # mode 0: w = max(B - 1, 0) = [[9,1],[0,3]]  -> sum 13
    s = oracle.threshold_cog(B, 0.1, 0)
    assert np.allclose(s, [((1 + 3) * 0.5 + 9 * -0.5) / 13, (3 * 0.5 + (9 + 1) * -0.5) / 13], atol=1e-15)
    # mode 1: w = B where B >= 1 -> [[10,2],[0,4]] -> sum 16
    s = oracle.threshold_cog(B, 0.1, 1)
    assert np.allclose(s, [((2 + 4) * 0.5 + 10 * -0.5) / 16, (4 * 0.5 + (10 + 2) * -0.5) / 16], atol=1e-15)


def test_I15_identity_cases(oracle):
    Sh = rng.random((16, 16))
    assert np.array_equal(oracle.bin_image(Sh, 1), Sh)
    want = Sh.reshape(4, 4, 4, 4).sum(axis=(1, 3))
    assert np.abs(oracle.bin_image(Sh, 4) - want).max() < 1e-14
    C = rng.random((8, 8))
    assert np.array_equal(oracle.centre(C), np.roll(C, (4, 4), (0, 1)))


# ---------------------------------------------------------------- I11, I12
@pytest.mark.parametrize("P", [8, 16, 32])
def test_I11_delta_kernels(oracle, P):
    I = rng.random((P, P))
    d = np.zeros((P, P), np.float32)
    d[P // 2, P // 2] = 1.0
    for direct in (False, True):
        assert np.abs(oracle.convolve(I, d, direct) - I).max() < 1e-13
        d2 = np.roll(d, (2, -3), (0, 1))
        assert np.abs(oracle.convolve(I, d2, direct) - np.roll(I, (2, -3), (0, 1))).max() < 1e-13


@pytest.mark.parametrize("P", [8, 16, 32])
def test_I12_fft_convolution_equals_direct_sum(oracle, P):
    I = rng.random((P, P))
    K = rng.random((P, P)).astype(np.float32)
    a = oracle.convolve(I, K, direct=False)
    c = oracle.convolve(I, K, direct=True)
    assert np.abs(a - c).max() < 1e-12 * np.abs(c).max()
    # and against numpy's transforms with the kernel recentred to the origin
    kc = np.roll(K.astype(np.float64), (-P // 2, -P // 2), (0, 1))
    lib = np.real(np.fft.ifft2(np.fft.fft2(I) * np.fft.fft2(kc)))
    assert np.abs(c - lib).max() < 1e-12 * np.abs(c).max()


# ---------------------------------------------------------------- I13
@pytest.mark.parametrize("n,P,b", SIZES)
def test_I13_wiener_khinchin(oracle, n, P, b):
    amp, yx = _one_sub(n, _partial_mask(n))
    ph = rng.normal(0, 2.0, (1, n, n)).astype(np.float32)
    _, Ic = oracle.measure(ph, amp, yx, n, P, b, stage=0)
    I = np.roll(Ic[0, 0], (-P // 2, -P // 2), (0, 1))                 # undo the centring
    e = oracle.field(ph[0], amp, n, P, 0, 0)[:n, :n]
    G = np.fft.fft2(I)                                                 # sum I exp(-2 pi i (v ly + u lx)/P)
    for ly in range(-(n - 1), n):
        for lx in range(-(n - 1), n):
            acc = 0.0
            for j in range(max(0, -ly), min(n, n - ly)):
                for k in range(max(0, -lx), min(n, n - lx)):
                    acc += e[j, k] * np.conj(e[j + ly, k + lx])
            assert abs(G[ly % P, lx % P] - acc) < 1e-11 * n * n
    if P >= 2 * n:                                                      # outside the support it vanishes
        assert abs(G[n, 0]) < 1e-11 * n * n and abs(G[0, n]) < 1e-11 * n * n


# ---------------------------------------------------------------- I16: numpy restatement of O1..O9
def _numpy_chain(ph, amp, yx, n, P, b, tau, K):
    T, nsub = ph.shape[0], len(yx)
    out = np.zeros((T, nsub, 2))
    D = P // b
    j, k = np.mgrid[0:n, 0:n]
    ref = (D - 1) / 2
    for t in range(T):
        for i, (sy, sx) in enumerate(yx):
            sl = np.s_[sy * n:(sy + 1) * n, sx * n:(sx + 1) * n]
            e = np.zeros((P, P), complex)
            e[:n, :n] = amp[sl] * np.exp(1j * (ph[t][sl].astype(np.float64) - np.pi * (j + k) / P))
            I = np.abs(np.fft.fft2(e)) ** 2 / P ** 2
            if K is not None:
                kc = np.roll(K[i].astype(np.float64), (-P // 2, -P // 2), (0, 1))
                I = np.real(np.fft.ifft2(np.fft.fft2(I) * np.fft.fft2(kc)))
            Sh = np.fft.fftshift(I)
            B = Sh.reshape(D, b, D, b).sum(axis=(1, 3))
            Wt = np.maximum(B - tau * B.max(), 0.0)
            R, Cc = np.mgrid[0:D, 0:D]
            out[t, i] = [(Wt * (Cc - ref)).sum() / Wt.sum(), (Wt * (R - ref)).sum() / Wt.sum()]
    return out


@pytest.mark.parametrize("cfg", [1, 2, 3, 5])
def test_I16_numpy_fft_restatement(oracle, cfg):
    c = W.CONFIGS[cfg]
    amp = W.pupil_mask(c)
    yx_all = oracle.valid_list(amp, c.n, c.min_illum)
    pick = np.linspace(0, len(yx_all) - 1, 24).astype(int)            # includes partially lit edge subaps
    yx = yx_all[pick]
    ph = W.phase_frames(c, 0, [0, 1])
    K = W.elongation_kernels(c, 0, yx_all, subset=pick)
    got = oracle.measure(ph, amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K)
    want = _numpy_chain(ph, amp, yx, c.n, c.P, c.b, c.tau, K)
    assert np.abs(got - want).max() < 1e-10
    assert np.abs(got).max() > 0.05                                    # not a trivial comparison


# ---------------------------------------------------------------- I17
def test_I17_geometry_counts(oracle):
    want = {1: (80, 60), 2: (1212, 1124), 3: (4632, 4440), 5: (4632, 4432)}
    for cfg, (nsub, nfull) in want.items():
        c = W.CONFIGS[cfg]
        amp = W.pupil_mask(c)
        yx = oracle.valid_list(amp, c.n, c.min_illum)
        assert len(yx) == nsub
        full = sum(1 for sy, sx in yx if amp[sy * c.n:(sy + 1) * c.n, sx * c.n:(sx + 1) * c.n].min() == 1.0)
        assert full == nfull
        assert np.all(np.diff(yx[:, 0] * c.S + yx[:, 1]) > 0)          # row-major, sy outer


def test_valid_list_by_hand(oracle):
    n = 2
    amp = np.zeros((4, 4), np.float32)
    amp[0:2, 0:2] = 1.0                  # (0,0): mean 1
    amp[0, 2] = amp[1, 3] = 1.0          # (0,1): mean 0.5 -> valid with >=
    amp[2, 0] = 1.0                      # (1,0): mean 0.25 -> invalid
    yx = oracle.valid_list(amp, n, 0.5)
    assert yx.tolist() == [[0, 0], [0, 1]]


def test_elongation_kernel_recipe_properties():
    """The harness kernels (A11): wrapped Gaussians are point-symmetric about (P/2,P/2) and sum to 1."""
    c = W.CONFIGS[3]
    amp = W.pupil_mask(c)
    from oracle import shwfs_oracle as O
    yx = O.valid_list(amp, c.n, c.min_illum)
    K = W.elongation_kernels(c, 2, yx, subset=[0, 2000, 4631]).astype(np.float64)
    idx = (c.P - np.arange(c.P)) % c.P
    for k in K:
        kc = np.roll(k, (-c.P // 2, -c.P // 2), (0, 1))
        assert np.abs(kc - kc[np.ix_(idx, idx)]).max() < 1e-9 * k.max()
        assert abs(k.sum() - 1.0) < 1e-6
    s_l, s_s, th = W.elongation_params(c, 2, yx)
    assert abs(s_l.max() - 21.81) < 0.01 and abs(s_s[0] - 5.45) < 0.01

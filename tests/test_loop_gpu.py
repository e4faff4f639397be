"""GPU <-> oracle parity of the closed-loop neighbours (shwfs_set_dm, shwfs_measure_residual,
shwfs_reconstruct, shwfs_closed_loop) through the C ABI, -m gpu."""
import numpy as np
import pytest

from paper_1408_0698_b200 import workloads as W

pytestmark = pytest.mark.gpu

SLOPE_TOL = 1e-3


@pytest.fixture(scope="module")
def loop():
    from oracle import closed_loop
    return closed_loop


def _wk_algos(s, B):
    out = []
    for a in (B.ALGO_WK, B.ALGO_WK_GENERIC, B.ALGO_WK_FFT):
        try:
            s.algorithm = a
            out.append(a)
        except B.ShwfsError as e:
            assert e.code == B.SHWFS_EUNSUPPORTED
    return out


@pytest.mark.parametrize("cfg_id,M,T", [(3, 13, 3), (1, 6, 37)])
def test_residual_slopes_match_oracle(gpu, oracle, loop, cfg_id, M, T):
    """Config 3 (MAORY LGS geometry, elongation kernels) with 13 modes (not a multiple of 4) and the tiny
    config with a ragged batch: slopes of open - DM against the oracle, every spot."""
    torch, B = gpu
    c = W.CONFIGS[cfg_id]
    amp = W.pupil_mask(c)
    yx = oracle.valid_list(amp, c.n, c.min_illum)
    K = W.elongation_kernels(c, 0, yx)
    modes = W.dm_modes(c, M)
    rng = np.random.default_rng(cfg_id)
    ph = W.phase_frames(c, 0, [t % 4 for t in range(T)])
    coef = rng.normal(0, 1.0, (T, M)).astype(np.float32)
    coef[:, :2] *= 0.3
    want = loop.measure_residual(ph, modes, coef, amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K)
    with B.from_config(c, 0, kernels=K, valid_yx=yx) as s:
        s.set_dm(torch.from_numpy(modes).cuda())
        phd, cd = torch.from_numpy(ph).cuda(), torch.from_numpy(coef).cuda()
        for a in _wk_algos(s, B):
            s.algorithm = a
            got = s.measure_residual(phd, cd).cpu().numpy()
            assert np.abs(got - want).max() <= SLOPE_TOL, (a, np.abs(got - want).max())
        # zero coefficients: the plain sensor
        s.algorithm = B.ALGO_WK
        z = s.measure_residual(phd, torch.zeros_like(cd)).cpu().numpy()
        np.testing.assert_allclose(z, s.measure(phd).cpu().numpy(), atol=1e-6)
        # dropping the DM
        s.set_dm(None)
        out = torch.empty((T, s.nsub, 2), dtype=torch.float32, device="cuda")
        assert B.load().shwfs_measure_residual(s._h, phd.data_ptr(), cd.data_ptr(), T, out.data_ptr(),
                                               None) == B.SHWFS_EINVAL


def test_reconstruct_matches_oracle(gpu, oracle, loop):
    torch, B = gpu
    c = W.CONFIGS[1]
    rng = np.random.default_rng(5)
    M, T = 7, 19
    with B.from_config(c, 0) as s:
        s.set_dm(torch.from_numpy(W.dm_modes(c, M)).cuda())
        R = rng.normal(0, 1, (M, 2 * s.nsub)).astype(np.float32)
        sl = rng.normal(0, 1, (T, s.nsub, 2)).astype(np.float32)
        c0 = rng.normal(0, 1, (T, M)).astype(np.float32)
        want = c0.astype(np.float64) + 0.4 * loop.reconstruct(R, sl)
        got = s.reconstruct(torch.from_numpy(R).cuda(), torch.from_numpy(sl).cuda(), torch.from_numpy(c0).cuda(),
                            gain=0.4).cpu().numpy()
        np.testing.assert_allclose(got, want, rtol=0, atol=2e-5 * np.abs(want).max())


@pytest.mark.parametrize("cfg_id,M,T,noise", [(3, 6, 5, False), (1, 5, 12, True)])
def test_closed_loop_matches_oracle(gpu, oracle, loop, cfg_id, M, T, noise):
    """T sequential frames: slopes, coefficient history and final coefficients against the oracle's loop;
    the control matrix is the pseudo-inverse of the oracle's push-pull interaction matrix (tiny config) or a
    seeded random matrix of small gain (config 3: parity only)."""
    torch, B = gpu
    c = W.CONFIGS[cfg_id]
    amp = W.pupil_mask(c)
    yx = oracle.valid_list(amp, c.n, c.min_illum)
    K = W.elongation_kernels(c, 0, yx)
    modes = W.dm_modes(c, M)
    rng = np.random.default_rng(10 + cfg_id)
    kw = dict(tau=c.tau, kernels=K)
    if cfg_id == 1:
        D = loop.interaction_matrix(modes, amp, yx, c.n, c.P, c.b, **kw)
        R = np.linalg.pinv(D)
        a_true = np.array([0.15, -0.1, 0.3, -0.2, 0.25])[:M]             # static, inside the DM's span: converges
        ph = np.repeat(np.einsum("m,myx->yx", a_true, modes.astype(np.float64))[None], T, axis=0).astype(np.float32)
    else:
        R = rng.normal(0, 1.0, (M, 2 * len(yx))) / len(yx)
        ph = W.phase_frames(c, 0, range(T))
    R = R.astype(np.float32)
    gain, c0 = 0.5, rng.normal(0, 0.1, M).astype(np.float32)
    want_s, want_h, want_c = loop.closed_loop(ph, modes, R, gain, c0, amp, yx, c.n, c.P, c.b, **kw)
    with B.from_config(c, 0, kernels=K, valid_yx=yx) as s:
        s.set_dm(torch.from_numpy(modes).cuda())
        cd = torch.from_numpy(c0.copy()).cuda()
        l0 = s.launch_count
        got_s, got_h = s.closed_loop(torch.from_numpy(ph).cuda(), torch.from_numpy(R).cuda(), gain, cd)
        assert s.launch_count - l0 == 3 * T
        scale = max(np.abs(want_h).max(), 1e-3)
        assert np.abs(got_s.cpu().numpy() - want_s).max() <= SLOPE_TOL
        np.testing.assert_allclose(got_h.cpu().numpy(), want_h, rtol=0, atol=2e-4 * scale)
        np.testing.assert_allclose(cd.cpu().numpy(), want_c, rtol=0, atol=2e-4 * scale)
        if cfg_id == 1:
            # the loop does correct: residual slopes shrink once the integrator has caught up
            assert np.abs(want_s[-1]).mean() < 0.7 * np.abs(want_s[0]).mean()
        if noise:
            # with detector noise frame t draws counter first_frame + t: same as T one-frame calls
            s.set_noise(50.0, 1.0, 7, first_frame=3)
            cd = torch.from_numpy(c0.copy()).cuda()
            phd, Rd = torch.from_numpy(ph).cuda(), torch.from_numpy(R).cuda()
            a_s, a_h = s.closed_loop(phd, Rd, gain, cd)
            ce = torch.from_numpy(c0.copy()).cuda()
            for t in range(T):
                s.set_noise(50.0, 1.0, 7, first_frame=3 + t)
                st = s.measure_residual(phd[t:t + 1], ce[None, :].contiguous())
                assert torch.equal(st[0], a_s[t])
                assert torch.equal(ce, a_h[t])
                cc = ce[None, :].contiguous()
                s.reconstruct(Rd, st, cc, gain)
                ce = cc[0]
            assert torch.equal(ce, cd)


def test_residual_with_sublayers(gpu, oracle):
    """DM + sodium sub-layers: the same DM phase is subtracted from every sub-layer's wavefront."""
    torch, B = gpu
    from oracle import closed_loop as loop
    c = W.CONFIGS[1]
    amp = W.pupil_mask(c)
    yx = oracle.valid_list(amp, c.n, c.min_illum)
    M, T, L = 5, 3, 2
    modes = W.dm_modes(c, M)
    rng = np.random.default_rng(3)
    ph = np.stack([W.phase_frames(c, 0, range(T)), W.phase_frames(c, 0, range(1, T + 1))], axis=1)
    coef = rng.normal(0, 0.5, (T, M)).astype(np.float32)
    w, de = np.array([0.6, 0.4]), np.array([0.3, -0.5])
    res = np.stack([loop.residual_phase(ph[:, l], modes, coef) for l in range(L)], axis=1).astype(np.float32)
    want = oracle.measure_lgs(res, amp, yx, c.n, c.P, c.b, c.dx, weight=w, defocus=de, cx=4.0, cy=0.0, tau=c.tau)
    with B.from_config(c, 0) as s:
        s.set_sodium(w, de, None, None, (4.0, 0.0))
        s.set_dm(torch.from_numpy(modes).cuda())
        for a in _wk_algos(s, B):
            s.algorithm = a
            got = s.measure_residual(torch.from_numpy(ph).cuda(), torch.from_numpy(coef).cuda()).cpu().numpy()
            assert np.abs(got - want).max() <= SLOPE_TOL, a


@pytest.mark.parametrize("cfg_id,M,T", [(3, 37, 20), (1, 50, 150), (5, 21, 12)])
def test_residual_batches_on_the_tensor_cores(gpu, oracle, loop, cfg_id, M, T):
    """Batches (T > 8) take the tcgen05 3xTF32 GEMM of dm_umma.cu (n*n = 100 -> N = 112, 64, 256; M not a
    multiple of the 16-mode stage; T = 150: two frame tiles, the second ragged): slopes against the oracle on a
    sample of subapertures, and against the FP32 SIMT GEMM (SHWFS_DM_FP32=1) on every spot."""
    import os
    torch, B = gpu
    c = W.CONFIGS[cfg_id]
    amp = W.pupil_mask(c)
    yx = oracle.valid_list(amp, c.n, c.min_illum)
    modes = W.dm_modes(c, M)
    rng = np.random.default_rng(100 + cfg_id)
    ph = W.phase_frames(c, 0, [t % 2 for t in range(T)])
    coef = rng.normal(0, 0.5, (T, M)).astype(np.float32)
    coef[:, :2] *= 0.3
    with B.from_config(c, 0) as s:
        s.set_dm(torch.from_numpy(modes).cuda())
        phd, cd = torch.from_numpy(ph).cuda(), torch.from_numpy(coef).cuda()
        l0 = s.launch_count
        got = s.measure_residual(phd, cd).cpu().numpy()
        assert s.launch_count - l0 == 3                     # split coefficients, tensor-core GEMM, sensor
        os.environ["SHWFS_DM_FP32"] = "1"
        try:
            ref = s.measure_residual(phd, cd).cpu().numpy()
        finally:
            del os.environ["SHWFS_DM_FP32"]
        assert np.abs(got - ref).max() <= 2e-5              # 3xTF32 is fp32-like: far inside the 1e-3 tolerance
        K = W.elongation_kernels(c, 0, yx)
        sel = np.sort(rng.choice(len(yx), size=min(len(yx), 60), replace=False))
        ts = [0, T // 2, T - 1]
        want = loop.measure_residual(ph[ts], modes, coef[ts], amp, yx[sel], c.n, c.P, c.b, tau=c.tau,
                                     kernels=None if K is None else K[sel])
        assert np.abs(got[ts][:, sel] - want).max() <= SLOPE_TOL


@pytest.mark.parametrize("n,P,b,T", [(5, 8, 1, 3), (12, 32, 2, 11), (6, 16, 1, 20), (14, 32, 2, 9)])
def test_residual_on_sizes_without_a_templated_gemm(gpu, oracle, loop, n, P, b, T):
    """Odd n (generic sensor kernel) and n*n outside {64, 100, 256}: the DM phase falls back to the
    one-thread-per-output kernel, for the loop step (T <= 8) and for batches alike."""
    torch, B = gpu
    S, N, M = 3, 3 * n, 7
    rng = np.random.default_rng(n * 10 + T)
    amp = (rng.random((N, N)) > 0.15).astype(np.float32)
    yx = np.array([[sy, sx] for sy in range(S) for sx in range(S)], dtype=np.int32)
    ph = rng.normal(0, 1.5, (T, N, N)).astype(np.float32)
    modes = rng.normal(0, 1.0, (M, N, N)).astype(np.float32)
    coef = rng.normal(0, 0.4, (T, M)).astype(np.float32)
    want = loop.measure_residual(ph, modes, coef, amp, yx, n, P, b, tau=0.1)
    with B.Shwfs(amp, S, n, 0.05, W.LAMBDA_M, P, b, valid_yx=yx, threshold_frac=0.1) as s:
        s.set_dm(torch.from_numpy(modes).cuda())
        got = s.measure_residual(torch.from_numpy(ph).cuda(), torch.from_numpy(coef).cuda()).cpu().numpy()
        assert np.abs(got - want).max() <= SLOPE_TOL
        R = rng.normal(0, 1, (M, 2 * len(yx))).astype(np.float32) / len(yx)
        ws, wh, wc = loop.closed_loop(ph[:4], modes, R, 0.4, np.zeros(M), amp, yx, n, P, b, tau=0.1)
        c0 = torch.zeros(M, device="cuda")
        gs, gh = s.closed_loop(torch.from_numpy(ph[:4]).cuda(), torch.from_numpy(R).cuda(), 0.4, c0)
        assert np.abs(gs.cpu().numpy() - ws).max() <= SLOPE_TOL
        np.testing.assert_allclose(c0.cpu().numpy(), wc, rtol=0, atol=2e-4 * max(np.abs(wc).max(), 1e-3))

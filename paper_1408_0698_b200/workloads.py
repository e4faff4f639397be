"""Seeded synthetic inputs for the Shack-Hartmann WFS hot path (numpy only).

This module serves BOTH the CUDA library and the CPU oracle with identical arrays and therefore holds
none of the method's arithmetic: it only makes *inputs* -- pupil amplitude masks, von Karman phase screens
and LGS elongation kernels -- with the shapes, sizes and statistics of the paper's MAORY workloads
("800x800 ... 4.875e-2 m"; "FFT from the Kolmogorov or Von Karman models of the
phase Power Spectrum"; "80x80 subapertures") and of BASELINE.json:configs.  The paper's own
.fits wavefront histories are not available; these stand in for them.

It imports neither the oracle nor the CUDA binding.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

ARCSEC = math.pi / (180.0 * 3600.0)
LAMBDA_M = 0.589e-6          # sensing wavelength, sodium line (BASELINE.json:configs[0])
R0_M = 0.15                  # Fried parameter at 0.5 um   (BASELINE.json:configs[0])
L0_M = 25.0                  # outer scale                 (BASELINE.json:configs[0])
SEED0 = 14080698


@dataclass(frozen=True)
class WfsConfig:
    """One row of the config table in SURVEY.md section 8 (BASELINE.json:configs[k-1])."""
    cfg: int            # 1..5
    name: str
    N: int              # pupil grid side
    dx: float           # metres per pupil pixel
    S: int              # subapertures per side
    n: int              # phase px per subaperture side
    P: int              # zero-padded FFT side
    b: int              # binning
    W: int              # number of WFS
    T: int              # frames per WFS
    batch: int          # frames per shwfs_measure call
    r_out: float        # pupil outer radius [m]
    r_in: float         # central obstruction radius [m]
    tau: float          # CoG threshold fraction
    elong_max_arcsec: float   # long-axis FWHM at the farthest subaperture; 0 = no elongation
    screen_M: int       # side of the FFT grid the screens are filtered on
    min_illum: float = 0.5
    fwhm_short_arcsec: float = 1.0

    @property
    def D(self) -> int:
        return self.P // self.b

    @property
    def pixel_scale_arcsec(self) -> float:
        """Unbinned focal-plane pixel, lambda / (P dx)."""
        return LAMBDA_M / (self.P * self.dx) / ARCSEC


CONFIGS = {
    1: WfsConfig(1, "tiny", 80, 0.10, 10, 8, 16, 1, 1, 4, 4, 4.0, 0.0, 0.0, 0.0, 256),
    2: WfsConfig(2, "8m", 640, 0.0125, 40, 16, 32, 2, 1, 100, 100, 4.0, 0.8, 0.10, 0.0, 1024),
    3: WfsConfig(3, "lgs1", 800, 0.04875, 80, 10, 32, 2, 1, 100, 100, 19.5, 5.5, 0.10, 4.0, 1024),
    4: WfsConfig(4, "lgs6", 800, 0.04875, 80, 10, 32, 2, 6, 1000, 100, 19.5, 5.5, 0.10, 4.0, 1024),
    5: WfsConfig(5, "stress", 1280, 0.030468750, 80, 16, 64, 4, 6, 1000, 100, 19.5, 5.5, 0.10, 6.0, 2048),
}


def seed_for(cfg: int, wfs: int, frame: int) -> int:
    """seed = 14080698 + 100000*cfg + 1000*wfs + frame."""
    return SEED0 + 100000 * cfg + 1000 * wfs + frame


def pupil_mask(c: WfsConfig) -> np.ndarray:
    """Reading A1: a[y,x] = 1 where r_in <= r <= r_out at the pixel centre, else 0 (fp32 [N,N])."""
    ax = (np.arange(c.N, dtype=np.float64) + 0.5 - c.N / 2.0) * c.dx
    r = np.hypot(ax[None, :], ax[:, None])
    return ((r >= c.r_in) & (r <= c.r_out)).astype(np.float32)


def _psd_filter(M: int, dx: float) -> np.ndarray:
    f = np.fft.fftfreq(M, dx)
    f2 = f[None, :] ** 2 + f[:, None] ** 2
    psd = 0.022896 * R0_M ** (-5.0 / 3.0) * (f2 + L0_M ** -2.0) ** (-11.0 / 6.0)
    psd[0, 0] = 0.0
    return np.sqrt(psd) / dx


_FILTERS: dict = {}


def phase_screen(c: WfsConfig, wfs: int, frame: int) -> np.ndarray:
    """One von Karman screen in radians at 0.589 um, fp32 [N,N] (recipe of SURVEY.md 8(d))."""
    key = (c.screen_M, c.dx)
    if key not in _FILTERS:
        _FILTERS[key] = _psd_filter(c.screen_M, c.dx)
    w = np.random.default_rng(seed_for(c.cfg, wfs, frame)).standard_normal((c.screen_M, c.screen_M))
    scr = np.real(np.fft.ifft2(np.fft.fft2(w) * _FILTERS[key]))
    scr *= 0.5 / 0.589
    return np.ascontiguousarray(scr[: c.N, : c.N], dtype=np.float32)


def phase_frames(c: WfsConfig, wfs: int, frames) -> np.ndarray:
    """Stack of screens [len(frames), N, N] fp32."""
    return np.stack([phase_screen(c, wfs, int(t)) for t in frames], axis=0)


def launch_point(c: WfsConfig, wfs: int):
    """Reading A13: launch telescope of WFS w at the pupil edge, 60 deg apart."""
    ang = math.radians(60.0 * wfs)
    return c.r_out * math.cos(ang), c.r_out * math.sin(ang)


def elongation_params(c: WfsConfig, wfs: int, valid_yx: np.ndarray):
    """Readings A11-A13: per-subaperture (sigma_long, sigma_short, theta) in unbinned pixels / radians."""
    yx = np.asarray(valid_yx, dtype=np.float64)
    yc = ((yx[:, 0] + 0.5) * c.n - c.N / 2.0) * c.dx
    xc = ((yx[:, 1] + 0.5) * c.n - c.N / 2.0) * c.dx
    lx, ly = launch_point(c, wfs)
    d = np.hypot(xc - lx, yc - ly)
    e_max = math.sqrt(c.elong_max_arcsec ** 2 - c.fwhm_short_arcsec ** 2)
    fwhm_l = np.sqrt(c.fwhm_short_arcsec ** 2 + (e_max * d / d.max()) ** 2)
    to_sigma = 1.0 / (2.0 * math.sqrt(2.0 * math.log(2.0))) / c.pixel_scale_arcsec
    theta = np.arctan2(yc - ly, xc - lx)
    return fwhm_l * to_sigma, np.full_like(d, c.fwhm_short_arcsec * to_sigma), theta


def elongation_kernels(c: WfsConfig, wfs: int, valid_yx: np.ndarray, subset=None, device=None,
                       chunk: int = 64):
    """Wrapped (periodically summed) rotated Gaussians, normalised to sum 1 in float64, cast to fp32.

    K_i[r,c] = sum_{m,l=-M..M} g(c-P/2+l*P, r-P/2+m*P),
    g(x,y) = exp(-((x cos t + y sin t)^2 / sL^2 + (-x sin t + y cos t)^2 / sS^2) / 2),  M = ceil(6 sL / P) + 1
    (readings A11-A13; the quadratic form is expanded to A x^2 + 2 B x y + C y^2 before the
    exponential, nothing else).  The per-subaperture parameters always come from the FULL valid list;
    `subset` (indices into it) restricts which kernels are evaluated.  Returns fp32 [len(subset),P,P]: a
    numpy array, or -- when `device` is a torch device -- a torch tensor on it (same formula in torch
    float64, for speed at the full sizes).  Returns None when the config has no elongation.
    """
    if c.elong_max_arcsec <= 0.0:
        return None
    s_l, s_s, th = elongation_params(c, wfs, valid_yx)
    P = c.P
    wraps = int(math.ceil(6.0 * float(s_l.max()) / P)) + 1
    if subset is not None:
        subset = np.asarray(subset, dtype=np.int64)
        s_l, s_s, th = s_l[subset], s_s[subset], th[subset]
    qa = 0.5 * (np.cos(th) ** 2 / s_l ** 2 + np.sin(th) ** 2 / s_s ** 2)       # exponent = -(qa x^2
    qc = 0.5 * (np.sin(th) ** 2 / s_l ** 2 + np.cos(th) ** 2 / s_s ** 2)       #   + qb x y + qc y^2)
    qb = np.cos(th) * np.sin(th) * (1.0 / s_l ** 2 - 1.0 / s_s ** 2)
    nw = 2 * wraps + 1
    ax_np = ((np.arange(P, dtype=np.float64) - P / 2.0)[None, :]
             + (np.arange(-wraps, wraps + 1, dtype=np.float64) * P)[:, None]).reshape(-1)
    if device is None:
        xp, ax = np, ax_np
        as_x = lambda a: np.asarray(a, dtype=np.float64)
        out = np.empty((len(s_l), P, P), dtype=np.float32)
    else:
        import torch
        xp = torch
        as_x = lambda a: torch.as_tensor(np.asarray(a, dtype=np.float64), device=device)
        ax = as_x(ax_np)
        out = torch.empty((len(s_l), P, P), dtype=torch.float32, device=device)
    xy = ax[None, :, None] * ax[None, None, :]                  # y (rows) times x (columns)
    x2 = (ax * ax)[None, None, :]
    y2 = (ax * ax)[None, :, None]
    for i0 in range(0, len(s_l), chunk):
        a_, b_, c_ = (as_x(q[i0:i0 + chunk])[:, None, None] for q in (qa, qb, qc))
        g = xy * b_
        g += x2 * a_
        g += y2 * c_
        g = xp.exp(-g)
        g = g.reshape(-1, nw, P, nw, P).sum(axis=3).sum(axis=1)   # periodic sum over image cells
        g = g / g.sum(axis=(1, 2)).reshape(-1, 1, 1)
        if xp is np:
            out[i0:i0 + chunk] = g.astype(np.float32)
        else:
            out[i0:i0 + chunk] = g.to(out.dtype)
    return out


def sodium_layers(c: WfsConfig, wfs: int, L: int, h0_m: float = 90e3, fwhm_m: float = 10e3):
    """Inputs of the paper's sub-layer model (reading B2): L equal slabs
    spanning +-fwhm_m about the focus altitude h0_m, at their mid altitudes h_l, with a Gaussian sodium
    profile of FWHM fwhm_m as weights (normalised to sum 1), defocus a_l = (pi/lambda)(1/h0 - 1/h_l)
    [rad/m^2] about the launch point of WFS `wfs`, and a seeded uplink tip-tilt of 0.05 arcsec rms per
    sub-layer [rad/m of phase gradient].  Returns a dict of float64 arrays / floats."""
    edges = np.linspace(-fwhm_m, fwhm_m, L + 1)
    dh = 0.5 * (edges[:-1] + edges[1:])
    h = h0_m + dh
    w = np.exp(-4.0 * math.log(2.0) * (dh / fwhm_m) ** 2)
    w = w / w.sum()
    a = (math.pi / LAMBDA_M) * (1.0 / h0_m - 1.0 / h)
    tt = np.random.default_rng(seed_for(c.cfg, wfs, 0) + 777).normal(0.0, 0.05 * ARCSEC, (2, L))
    cx, cy = launch_point(c, wfs)
    return dict(weight=w, defocus=a, tilt_x=tt[0] * 2.0 * math.pi / LAMBDA_M,
                tilt_y=tt[1] * 2.0 * math.pi / LAMBDA_M, cx=cx, cy=cy, altitude=h)


def spot_size_kernels(c: WfsConfig, valid_yx: np.ndarray, device=None):
    """Round Gaussian of FWHM fwhm_short_arcsec for every subaperture (the laser-spot size; with sub-layers
    the elongation comes from the geometry).  Same evaluation as elongation_kernels."""
    from dataclasses import replace
    return elongation_kernels(replace(c, elong_max_arcsec=c.fwhm_short_arcsec * (1.0 + 1e-9)), 0, valid_yx,
                              device=device)


def dm_modes(c: WfsConfig, M: int) -> np.ndarray:
    """Stand-in for the paper's modal base (Zernike or Karhunen-Loeve modes fitted by the
    actuators): mode 0 and 1 are x and y tilt of one unbinned pixel of spot motion (2 pi / P rad per pupil
    pixel); the others are seeded von Karman screens (same recipe as phase_screen, seeds of "WFS" 900+m)
    scaled to 1 rad rms over the pupil -- smooth, turbulence-like shapes.  fp32 [M,N,N]."""
    amp = pupil_mask(c) > 0
    ax = np.arange(c.N, dtype=np.float64) + 0.5 - c.N / 2.0
    out = np.empty((M, c.N, c.N), dtype=np.float32)
    for m in range(M):
        if m == 0:
            md = np.broadcast_to(ax[None, :] * (2.0 * math.pi / c.P), (c.N, c.N))
        elif m == 1:
            md = np.broadcast_to(ax[:, None] * (2.0 * math.pi / c.P), (c.N, c.N))
        else:
            md = phase_screen(c, 900 + m, 0).astype(np.float64)
            md = md - md[amp].mean()
            md = md / md[amp].std()
        out[m] = md
    return out


def dm_modes_device(c: WfsConfig, M: int, device):
    """dm_modes with the screens generated on `device` (phase_frames_device, "WFS" 900): timing runs only."""
    import torch
    out = torch.empty((M, c.N, c.N), dtype=torch.float32, device=device)
    ax = (torch.arange(c.N, dtype=torch.float64, device=device) + 0.5 - c.N / 2.0) * (2.0 * math.pi / c.P)
    out[0] = ax[None, :].expand(c.N, c.N).to(torch.float32)
    if M > 1:
        out[1] = ax[:, None].expand(c.N, c.N).to(torch.float32)
    if M > 2:
        phase_frames_device(c, 900, range(2, M), device, out=out[2:])
        amp = torch.as_tensor(pupil_mask(c) > 0, device=device)
        for m in range(2, M):
            v = out[m][amp]
            out[m] = (out[m] - v.mean()) / v.std()
    return out


@dataclass(frozen=True)
class PyramidConfig:
    """Pyramid-WFS workload.  PAPER.md:96 describes the paper's pyramid test case on the
    LBT: "a 400 modes correction using a modulated (3 lambda/D) pyramid on a seeing of 1 arcsec"; the LBT
    pyramid has 30 x 30 subapertures on an 8.2 m pupil with an 11 % central obstruction."""
    name: str
    N: int              # pupil grid side (the pupil diameter spans it)
    dx: float           # metres per pupil pixel
    Np: int             # padded transform side
    s: int              # pupil-copy separation
    bp: int             # pupil pixels per detector pixel
    r_mod: float        # lambda / D
    K: int              # modulation points
    obstruction: float  # linear central obstruction
    screen_cfg: int     # WfsConfig whose screen recipe (grid, seeds) the frames come from

    @property
    def D_pix(self) -> float:
        return float(self.N)


PYRAMIDS = {
    "tiny": PyramidConfig("tiny", 48, 0.17, 256, 64, 4, 3.0, 8, 0.11, 1),
    "lbt": PyramidConfig("lbt", 240, 8.2 / 240, 1024, 256, 8, 3.0, 16, 0.11, 2),
}


def pyramid_mask(p: PyramidConfig) -> np.ndarray:
    ax = np.arange(p.N, dtype=np.float64) + 0.5 - p.N / 2.0
    r = np.hypot(ax[None, :], ax[:, None])
    return ((r <= p.N / 2.0) & (r >= p.obstruction * p.N / 2.0)).astype(np.float32)


def pyramid_frames(p: PyramidConfig, frames, scale: float = 1.0) -> np.ndarray:
    """Seeded von Karman frames for the pyramid ([T,N,N] fp32): the screen recipe of config `screen_cfg`
    (phase_screen, "WFS" 800), cropped to N x N and multiplied by `scale` (closed-loop residuals are a
    fraction of the open-loop turbulence)."""
    c = CONFIGS[p.screen_cfg]
    return np.stack([phase_screen(c, 800, int(t))[: p.N, : p.N] * np.float32(scale) for t in frames], axis=0)


def phase_frames_device(c: WfsConfig, wfs: int, frames, device, out=None):
    """Same von Karman recipe as phase_screen, evaluated with torch on `device` (float64 FFT, cast to fp32).

    The noise comes from torch's generator seeded with seed_for(cfg, wfs, frame), so the values differ from
    the numpy screens while the spectrum, variance and range are the same.  Used for the full-size timing
    runs only (throughput does not depend on the values); parity inputs come from
    phase_screen.  Returns a float32 tensor [len(frames), N, N] on `device` (written into `out` if given).
    """
    import torch
    frames = list(frames)
    filt = torch.as_tensor(_psd_filter(c.screen_M, c.dx), device=device)
    if out is None:
        out = torch.empty((len(frames), c.N, c.N), dtype=torch.float32, device=device)
    gen = torch.Generator(device=device)
    for q, t in enumerate(frames):
        gen.manual_seed(seed_for(c.cfg, wfs, int(t)))
        w = torch.randn((c.screen_M, c.screen_M), dtype=torch.float64, device=device, generator=gen)
        scr = torch.fft.ifft2(torch.fft.fft2(w) * filt).real * (0.5 / 0.589)
        out[q] = scr[: c.N, : c.N].to(torch.float32)
    return out

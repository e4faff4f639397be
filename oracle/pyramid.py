"""float64 CPU oracle of the pyramid wavefront sensor.

TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It imports nothing from the CUDA package and shares no code
with it.  Plain numpy in float64; numpy.fft.fft2 / ifft2 serve as the two transform steps (pinned against a
brute-force DFT in tests/test_oracle_pyramid_pins.py), everything else is written out step by step.

Passage followed, PAPER.md:92 (section 4, "Pyramid WFS"):
    "We follow the scheme presented in (Verinaud 2004), see also [15].  This module makes a large use of the
     GPU computing power for the whole computation including matrix-matrix complex array multiplications, Fast
     Fourier Transform and other operations on arrays."
and PAPER.md:96 ("a modulated (3 lambda/D) pyramid").  The paper gives no formula; the steps below are the
standard Fourier-optics model of that reference (readings D1..D7):

  Q1 field        e_k[y,x] = a[y,x] * exp(i*(c_phi*phi[y,x] + 2*pi*r_mod*(x*cos(th_k) + y*sin(th_k))/D_pix)),
                  th_k = 2*pi*(k + 1/2)/K, k < K modulation points on a circle of radius r_mod [lambda/D],
                  D_pix the pupil diameter in pixels, x, y the pixel indices; zero elsewhere on Np x Np
                  (pupil in the corner [0,N)^2).  K == 0 or r_mod == 0: one unmodulated point.
  Q2 focal plane  F_k = DFT2(e_k), forward, exp(-2*pi*i*...), unnormalised.
  Q3 pyramid      F_k *= exp(-2*pi*i * s * (|u~| + |v~|) / Np),  u~ = u if u < Np/2 else u - Np (signed
                  frequency index; the apex sits on the unaberrated spot), s = separation in pixels: the four
                  faces send the light to four copies of the pupil displaced by (+-s, +-s).
  Q4 pupil plane  G_k = IDFT2(F_k) (with the 1/Np^2), I_k = |G_k|^2.
  Q5 modulation   I = (1/K) sum_k I_k.
  Q6 quadrants    Q[a][b][y,x] = I[(y + a*s) mod Np, (x + b*s) mod Np], a, b in {+1,-1}, y, x < N; binned by
                  bp x bp block sums to Sp x Sp detector pixels (N = Sp*bp).
  Q7 signals      for each valid detector pixel i = (Y,X) (valid: mean pupil amplitude over its block >=
                  min_illum, row-major):  tot = Q++ + Q+- + Q-+ + Q--;  I0 = mean of tot over the valid pixels;
                  s_x[i] = (Q[+][+] + Q[-][+] - Q[+][-] - Q[-][-]) / I0   (b = +1 minus b = -1: light thrown
                  towards +x counts positive), s_y[i] with a.  Output [nvalid, 2] = (s_x, s_y).
                  Sign: a wavefront whose phase grows with x sends the spot to u~ > 0, i.e. to b = +1: s_x > 0.
"""
from __future__ import annotations

import numpy as np


def valid_pixels(amplitude, bp, min_illum=0.5):
    """Q7 validity rule: detector pixels whose bp x bp block of the pupil has mean amplitude >= min_illum."""
    a = np.asarray(amplitude, dtype=np.float64)
    N = a.shape[0]
    Sp = N // bp
    m = a.reshape(Sp, bp, Sp, bp).mean(axis=(1, 3))
    yx = np.argwhere(m >= min_illum).astype(np.int32)
    return yx


def field(phase, amplitude, Np, r_mod, theta, D_pix, c_phi=1.0):
    """Q1 for one modulation angle theta (r_mod = 0: no tilt)."""
    ph = np.asarray(phase, dtype=np.float64)
    a = np.asarray(amplitude, dtype=np.float64)
    N = ph.shape[0]
    y, x = np.mgrid[0:N, 0:N].astype(np.float64)
    arg = c_phi * ph + 2.0 * np.pi * r_mod * (x * np.cos(theta) + y * np.sin(theta)) / D_pix
    e = np.zeros((Np, Np), dtype=np.complex128)
    e[:N, :N] = a * np.exp(1j * arg)
    return e


def pyramid_mask(Np, s):
    """Q3: exp(-2 pi i s (|u~| + |v~|) / Np) on the DFT index grid."""
    u = np.arange(Np)
    us = np.where(u < Np // 2, u, u - Np).astype(np.float64)
    return np.exp(-2j * np.pi * s * (np.abs(us)[None, :] + np.abs(us)[:, None]) / Np)


def detector_intensity(phase, amplitude, Np, s, r_mod, K, D_pix, c_phi=1.0):
    """Q1..Q5: modulation-averaged intensity on the Np x Np pupil-plane grid."""
    mask = pyramid_mask(Np, s)
    if K <= 0 or r_mod == 0.0:
        thetas, r = [0.0], 0.0
    else:
        thetas, r = [2.0 * np.pi * (k + 0.5) / K for k in range(K)], r_mod
    I = np.zeros((Np, Np), dtype=np.float64)
    for th in thetas:
        F = np.fft.fft2(field(phase, amplitude, Np, r, th, D_pix, c_phi))        # Q2
        G = np.fft.ifft2(F * mask)                                                # Q3, Q4
        I += G.real ** 2 + G.imag ** 2
    return I / len(thetas)                                                        # Q5


def quadrants(I, N, s, bp):
    """Q6: the four pupil copies, binned.  Returns Q[a_index][b_index][Sp,Sp], index 0 = +1, 1 = -1."""
    Np = I.shape[0]
    Sp = N // bp
    out = np.zeros((2, 2, Sp, Sp), dtype=np.float64)
    idx = np.arange(N)
    for ia, a in enumerate((+1, -1)):
        for ib, b in enumerate((+1, -1)):
            q = I[np.ix_((idx + a * s) % Np, (idx + b * s) % Np)]
            out[ia, ib] = q.reshape(Sp, bp, Sp, bp).sum(axis=(1, 3))
    return out


def signals(Q, valid_yx):
    """Q7: (s_x, s_y) per valid detector pixel, normalised by the mean total intensity."""
    yx = np.asarray(valid_yx)
    q = Q[:, :, yx[:, 0], yx[:, 1]]                      # [2,2,nvalid]
    tot = q.sum(axis=(0, 1))
    I0 = tot.mean()
    sx = (q[0, 0] + q[1, 0] - q[0, 1] - q[1, 1]) / I0
    sy = (q[0, 0] + q[0, 1] - q[1, 0] - q[1, 1]) / I0
    return np.stack([sx, sy], axis=1)


def measure(phase, amplitude, valid_yx, Np, s, bp, r_mod, K, D_pix, c_phi=1.0, return_quadrants=False):
    """Q1..Q7 for every frame: phase [T,N,N] -> signals [T,nvalid,2] float64 (and Q [T,2,2,Sp,Sp])."""
    ph = np.asarray(phase)
    if ph.ndim == 2:
        ph = ph[None]
    N = ph.shape[-1]
    out, qs = [], []
    for t in range(ph.shape[0]):
        I = detector_intensity(ph[t], amplitude, Np, s, r_mod, K, D_pix, c_phi)
        Q = quadrants(I, N, s, bp)
        qs.append(Q)
        out.append(signals(Q, valid_yx))
    return (np.stack(out), np.stack(qs)) if return_quadrants else np.stack(out)

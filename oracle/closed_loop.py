"""float64 CPU oracle of the closed-loop neighbours of the Shack-Hartmann path.

TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It imports nothing from the CUDA package and shares no code
with it.  Plain numpy in float64, one function per sentence of the passage, in the paper's order.

Passage followed, PAPER.md:76 (section 3, "The closed loop"):
    "The WFS modules compute the vector signals (X-and Y- slopes) from the residual phase (the open loop
     wavefront subtracted by the DM).  Vector slopes multiplied by the control matrix returns the vector
     coefficients for the modal base linear composition, in the form of the differential coefficients to be
     added to the one defining the existing mirror shape.  [...] At this stage we consider a pure integrator
     scheme for the loop control."
and PAPER.md:68 ("the deformable mirrors are computed as the linear combination of a modal base"),
PAPER.md:69 (interaction matrix: "The modes defined in the base in input are used to register the slope
measured by the WFS modules"), PAPER.md:75 (control matrix = pseudo-inverse of the interaction matrix).

Readings (C1..C4; the paper gives no formula):
  C1  DM phase of frame t = sum_m c[t,m] * mode[m] (same units as the wavefront); residual = open - DM.
  C2  slope vector of a frame: s[k], k = 2*i + axis (x then y per valid subaperture, the layout of
      slopes[t,i,:]); differential coefficients d[m] = sum_k R[m,k] * s[k].
  C3  pure integrator: c_{t+1} = c_t + gain * d_t, where d_t comes from the slopes of the residual
      open_t - DM(c_t): the correction computed on frame t acts from frame t+1 (one frame of delay).
  C4  history convention: hist[t] = c_t, the coefficients that shaped the mirror for frame t; the function
      returns c_T as well.

Pins (tests/test_oracle_loop_pins.py): K1 zero coefficients leave the wavefront untouched; K2 a wavefront
that IS a mode combination is cancelled exactly (flat residual -> zero slopes); K3 residual and
reconstruction against their numpy einsum restatement on random inputs, including the k = 2i + axis order;
K4 a static tilt under a tilt-mode DM with the control matrix built by push-pull converges as
(1 - gain)^t (closed form of the pure integrator: sign, delay and update order); K5 gain = 0 freezes the
mirror, a wrong-sign control matrix diverges.
"""
from __future__ import annotations

import numpy as np

from . import shwfs_oracle as O


def residual_phase(open_phase, modes, coef):
    """C1: residual[t] = open[t] - sum_m coef[t,m] * modes[m], float64 [T,N,N]."""
    ph = np.asarray(open_phase, dtype=np.float64)
    md = np.asarray(modes, dtype=np.float64)
    c = np.asarray(coef, dtype=np.float64)
    T, M = c.shape
    res = ph.copy()
    for t in range(T):
        for m in range(M):
            res[t] -= c[t, m] * md[m]
    return res


def reconstruct(R, slopes):
    """C2: d[t,m] = sum_k R[m,k] * s[t,k] with k = 2*i + axis; slopes [T,nsub,2] -> [T,M] float64."""
    R = np.asarray(R, dtype=np.float64)
    s = np.asarray(slopes, dtype=np.float64)
    T = s.shape[0]
    flat = s.reshape(T, -1)
    out = np.zeros((T, R.shape[0]), dtype=np.float64)
    for t in range(T):
        out[t] = R @ flat[t]
    return out


def measure_residual(open_phase, modes, coef, amplitude, valid_yx, n, P, b, **wfs_kw):
    """Slopes of the residual phase (first sentence).  The residual is formed in float64 and
    handed to the Shack-Hartmann oracle, whose input type is fp32, rounded once."""
    res = residual_phase(open_phase, modes, coef).astype(np.float32)
    return O.measure(res, amplitude, valid_yx, n, P, b, **wfs_kw)


def closed_loop(open_phase, modes, R, gain, coef0, amplitude, valid_yx, n, P, b, **wfs_kw):
    """C3/C4: T sequential frames of the pure-integrator loop.

    Returns (slopes [T,nsub,2], hist [T,M] with hist[t] = c_t, c_T)."""
    ph = np.asarray(open_phase)
    T = ph.shape[0]
    c = np.array(coef0, dtype=np.float64).copy()
    M = c.shape[0]
    hist = np.zeros((T, M), dtype=np.float64)
    slopes = []
    for t in range(T):
        hist[t] = c
        s = measure_residual(ph[t:t + 1], modes, c[None, :], amplitude, valid_yx, n, P, b, **wfs_kw)
        slopes.append(s[0])
        d = reconstruct(R, s)[0]
        c = c + gain * d
    return np.stack(slopes, axis=0), hist, c


def interaction_matrix(modes, amplitude, valid_yx, n, P, b, amp_push=0.05, **wfs_kw):
    """PAPER.md:69 / :113 push-pull calibration: column m = (s(+a mode_m) - s(-a mode_m)) / (2a) with a flat
    incoming wavefront.  Returns D [2*nsub, M] float64 (the WFS sees open - DM, so pushing the MIRROR by +a
    gives slopes of -a*mode; the matrix is defined on the wavefront side: slopes per unit of +mode in the
    wavefront)."""
    md = np.asarray(modes, dtype=np.float64)
    M = md.shape[0]
    cols = []
    for m in range(M):
        push = (amp_push * md[m]).astype(np.float32)[None]
        sp = O.measure(push, amplitude, valid_yx, n, P, b, **wfs_kw)[0].reshape(-1)
        sm = O.measure(-push, amplitude, valid_yx, n, P, b, **wfs_kw)[0].reshape(-1)
        cols.append((sp - sm) / (2.0 * amp_push))
    return np.stack(cols, axis=1)

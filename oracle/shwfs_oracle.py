"""ctypes front end of the float64 CPU oracle (oracle/shwfs_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
imports nothing from paper_1408_0698_b200 and shares no code with the CUDA path.

Every function is a thin marshalling layer over one C function whose header
comment cites the passage it follows (PAPER.md:91 and the O1..O9 steps of
SURVEY.md 8(c)); there is no arithmetic of the method in this file.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "shwfs_oracle.c"
_SRCS = [_SRC, _HERE / "shwfs_oracle_lgs.c", _HERE / "shwfs_oracle_poisson.c"]
_LIB = _HERE / "libshwfs_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile shwfs_oracle.c -> libshwfs_oracle.so with gcc -O2 -fopenmp (the oracle as it stands)."""
    if force or not _LIB.exists() or any(_LIB.stat().st_mtime < f.stat().st_mtime for f in _SRCS):
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", str(tmp), *map(str, _SRCS), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


_f32p = np.ctypeslib.ndpointer(dtype=np.float32, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_i32p = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        L.shwfs_oracle_field.argtypes = [_f32p, _f32p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                                         C.c_double, _f64p]
        L.shwfs_oracle_field.restype = None
        L.shwfs_oracle_dft1.argtypes = [_f64p, _f64p, C.c_int, C.c_int]
        L.shwfs_oracle_dft1.restype = None
        L.shwfs_oracle_dft2.argtypes = [_f64p, _f64p, C.c_int, C.c_int]
        L.shwfs_oracle_dft2.restype = C.c_int
        L.shwfs_oracle_dft2_brute.argtypes = [_f64p, _f64p, C.c_int, C.c_int]
        L.shwfs_oracle_dft2_brute.restype = None
        L.shwfs_oracle_intensity.argtypes = [_f64p, C.c_int, _f64p]
        L.shwfs_oracle_intensity.restype = None
        L.shwfs_oracle_convolve_direct.argtypes = [_f64p, _f32p, C.c_int, _f64p]
        L.shwfs_oracle_convolve_direct.restype = None
        L.shwfs_oracle_convolve_fft.argtypes = [_f64p, _f32p, C.c_int, _f64p]
        L.shwfs_oracle_convolve_fft.restype = C.c_int
        L.shwfs_oracle_centre.argtypes = [_f64p, C.c_int, _f64p]
        L.shwfs_oracle_centre.restype = None
        L.shwfs_oracle_bin.argtypes = [_f64p, C.c_int, C.c_int, _f64p]
        L.shwfs_oracle_bin.restype = None
        L.shwfs_oracle_threshold_cog.argtypes = [_f64p, C.c_int, C.c_double, C.c_int, _f64p]
        L.shwfs_oracle_threshold_cog.restype = None
        L.shwfs_oracle_valid_list.argtypes = [_f32p, C.c_int, C.c_int, C.c_double, C.c_void_p]
        L.shwfs_oracle_valid_list.restype = C.c_int
        L.shwfs_oracle_measure.argtypes = [_f32p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, _f32p, _i32p,
                                           C.c_int, C.c_double, C.c_double, C.c_int, C.c_void_p, C.c_int,
                                           _f64p, C.c_int, C.c_void_p, C.c_int]
        L.shwfs_oracle_measure.restype = C.c_int
        L.shwfs_oracle_max_threads.argtypes = []
        L.shwfs_oracle_max_threads.restype = C.c_int
        u32p = np.ctypeslib.ndpointer(dtype=np.uint32, flags="C_CONTIGUOUS")
        L.shwfs_oracle_field_layer.argtypes = [_f32p, _f32p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int] + \
            [C.c_double] * 7 + [_f64p]
        L.shwfs_oracle_field_layer.restype = None
        L.shwfs_oracle_philox4x32.argtypes = [u32p, u32p, u32p]
        L.shwfs_oracle_philox4x32.restype = None
        L.shwfs_oracle_normal4.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, _f64p]
        L.shwfs_oracle_normal4.restype = None
        L.shwfs_oracle_add_noise.argtypes = [_f64p, C.c_int, C.c_double, C.c_double, C.c_uint64, C.c_uint32,
                                             C.c_uint32, _f64p]
        L.shwfs_oracle_add_noise.restype = None
        L.shwfs_oracle_measure_lgs.argtypes = [_f32p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                                               _f32p, _i32p, C.c_int, C.c_double, C.c_double, _f64p, _f64p,
                                               _f64p, _f64p, C.c_double, C.c_double, C.c_double, C.c_int,
                                               C.c_void_p, C.c_double, C.c_double, C.c_uint64, _f64p, C.c_int,
                                               C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L.shwfs_oracle_measure_lgs.restype = C.c_int
        L.shwfs_oracle_poisson_uniforms.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, _f64p]
        L.shwfs_oracle_poisson_uniforms.restype = None
        L.shwfs_oracle_poisson_inversion.argtypes = [C.c_double, C.c_double, C.POINTER(C.c_double)]
        L.shwfs_oracle_poisson_inversion.restype = C.c_long
        L.shwfs_oracle_poisson_draw.argtypes = [C.c_double, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32,
                                                C.POINTER(C.c_double)]
        L.shwfs_oracle_poisson_draw.restype = C.c_long
        L.shwfs_oracle_add_noise_poisson.argtypes = [_f64p, C.c_int, C.c_double, C.c_double, C.c_uint64, C.c_uint32,
                                                     C.c_uint32, _f64p, C.c_void_p]
        L.shwfs_oracle_add_noise_poisson.restype = None
        _lib = L
    return _lib


def _c(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def _cplx_in(z, P):
    z = np.ascontiguousarray(z, dtype=np.complex128).reshape(P, P)
    return z.view(np.float64).reshape(P, 2 * P)


def field(phase_frame, amplitude, n, P, sy, sx, c_phi=1.0):
    """O1+O2: complex P x P field of subaperture (sy,sx) (patch in the corner, zero padded)."""
    ph = _c(phase_frame, np.float32)
    am = _c(amplitude, np.float32)
    N = ph.shape[-1]
    out = np.zeros((P, 2 * P), dtype=np.float64)
    lib().shwfs_oracle_field(ph, am, N, n, P, sy, sx, float(c_phi), out)
    return out.view(np.complex128).reshape(P, P)


def dft1(x, sign=-1):
    x = np.ascontiguousarray(x, dtype=np.complex128)
    L = x.shape[0]
    out = np.zeros(2 * L, dtype=np.float64)
    lib().shwfs_oracle_dft1(x.view(np.float64), out, L, sign)
    return out.view(np.complex128)


def dft2(x, sign=-1):
    """O3: unnormalised 2-D DFT with exp(sign*2*pi*i*...) (naive for P<=16, radix-2 above)."""
    P = x.shape[0]
    out = np.zeros((P, 2 * P), dtype=np.float64)
    rc = lib().shwfs_oracle_dft2(_cplx_in(x, P), out, P, sign)
    if rc:
        raise MemoryError("oracle dft2")
    return out.view(np.complex128).reshape(P, P)


def dft2_brute(x, sign=-1):
    P = x.shape[0]
    out = np.zeros((P, 2 * P), dtype=np.float64)
    lib().shwfs_oracle_dft2_brute(_cplx_in(x, P), out, P, sign)
    return out.view(np.complex128).reshape(P, P)


def intensity(E):
    """O4: |E|^2 / P^2."""
    P = E.shape[0]
    out = np.zeros((P, P), dtype=np.float64)
    lib().shwfs_oracle_intensity(_cplx_in(E, P), P, out)
    return out


def convolve(I, K, direct=False):
    """O5: circular convolution, kernel centre at (P/2, P/2)."""
    I = _c(I, np.float64)
    K = _c(K, np.float32)
    P = I.shape[0]
    out = np.zeros((P, P), dtype=np.float64)
    if direct:
        lib().shwfs_oracle_convolve_direct(I, K, P, out)
    elif lib().shwfs_oracle_convolve_fft(I, K, P, out):
        raise MemoryError("oracle convolve")
    return out


def centre(Cimg):
    """O6: roll by P/2 on both axes."""
    Cimg = _c(Cimg, np.float64)
    P = Cimg.shape[0]
    out = np.zeros((P, P), dtype=np.float64)
    lib().shwfs_oracle_centre(Cimg, P, out)
    return out


def bin_image(Sh, b):
    """O7: b x b block sums."""
    Sh = _c(Sh, np.float64)
    P = Sh.shape[0]
    D = P // b
    out = np.zeros((D, D), dtype=np.float64)
    lib().shwfs_oracle_bin(Sh, P, b, out)
    return out


def threshold_cog(B, tau=0.0, mode=0):
    """O8+O9: thresholded centre of gravity, returns (s_x, s_y) in detector pixels."""
    B = _c(B, np.float64)
    D = B.shape[0]
    out = np.zeros(2, dtype=np.float64)
    lib().shwfs_oracle_threshold_cog(B, D, float(tau), int(mode), out)
    return out


def valid_list(amplitude, n, min_illum=0.5):
    """H0 / reading A2: (sy,sx) of subapertures with mean amplitude >= min_illum, row-major."""
    am = _c(amplitude, np.float32)
    N = am.shape[0]
    S = N // n
    yx = np.zeros((S * S, 2), dtype=np.int32)
    cnt = lib().shwfs_oracle_valid_list(am, N, n, float(min_illum), yx.ctypes.data_as(C.c_void_p))
    return yx[:cnt].copy()


def max_threads() -> int:
    return int(lib().shwfs_oracle_max_threads())


def measure(phase, amplitude, valid_yx, n, P, b, *, c_phi=1.0, tau=0.0, mode=0, kernels=None,
            conv_direct=False, stage=-1, nthreads=0):
    """O1..O9 for every frame and valid subaperture.

    phase [T,N,N] fp32, amplitude [N,N] fp32, valid_yx [nsub,2] int32, kernels [nsub,P,P] fp32 or None.
    Returns slopes [T,nsub,2] float64, or (slopes, images) if stage in {0,1,2}:
    0 = centred intensity [T,nsub,P,P], 1 = centred convolved image, 2 = binned image [T,nsub,D,D].
    """
    ph = _c(phase, np.float32)
    if ph.ndim == 2:
        ph = ph[None]
    T, N, _ = ph.shape
    am = _c(amplitude, np.float32)
    yx = _c(valid_yx, np.int32)
    nsub = yx.shape[0]
    slopes = np.zeros((T, nsub, 2), dtype=np.float64)
    kptr = None
    if kernels is not None:
        kernels = _c(kernels, np.float32)
        assert kernels.shape == (nsub, P, P), kernels.shape
        kptr = kernels.ctypes.data_as(C.c_void_p)
    images = None
    iptr = None
    if stage >= 0:
        D = P // b
        shp = (T, nsub, D, D) if stage == 2 else (T, nsub, P, P)
        images = np.zeros(shp, dtype=np.float64)
        iptr = images.ctypes.data_as(C.c_void_p)
    rc = lib().shwfs_oracle_measure(ph, T, N, n, P, b, am, yx, nsub, float(c_phi), float(tau), int(mode),
                                    kptr, int(bool(conv_direct)), slopes, int(stage), iptr, int(nthreads))
    if rc:
        raise RuntimeError(f"shwfs_oracle_measure failed with code {rc}")
    return (slopes, images) if stage >= 0 else slopes


# ---- paper's full LGS model: sodium sub-layers (f1) and detector noise (f2), oracle/shwfs_oracle_lgs.c ----

def field_layer(phase_frame, amplitude, n, P, sy, sx, dx, *, c_phi=1.0, defocus=0.0, cx=0.0, cy=0.0,
                tilt_x=0.0, tilt_y=0.0):
    """L1: complex P x P field of one sodium sub-layer (wavefront + a|r-r_c|^2 + g.r)."""
    ph = _c(phase_frame, np.float32)
    am = _c(amplitude, np.float32)
    N = ph.shape[-1]
    out = np.zeros((P, 2 * P), dtype=np.float64)
    lib().shwfs_oracle_field_layer(ph, am, N, n, P, sy, sx, float(c_phi), float(dx), float(defocus), float(cx),
                                   float(cy), float(tilt_x), float(tilt_y), out)
    return out.view(np.complex128).reshape(P, P)


def philox4x32(ctr, key):
    """L5: one Philox4x32-10 block; ctr = 4 uint32, key = 2 uint32 -> 4 uint32."""
    out = np.zeros(4, dtype=np.uint32)
    lib().shwfs_oracle_philox4x32(_c(ctr, np.uint32), _c(key, np.uint32), out)
    return out


def normal4(seed, t, i, blk):
    """L5: the four N(0,1) deviates of Philox block `blk` of spot (t, i)."""
    z = np.zeros(4, dtype=np.float64)
    lib().shwfs_oracle_normal4(int(seed), int(t), int(i), int(blk), z)
    return z


def add_noise(B, F, ron, seed, t, i):
    """L4: counts = F*B + sqrt(max(F*B,0)+ron^2)*z on a D x D binned image (F <= 0: unchanged)."""
    B = _c(B, np.float64)
    out = np.zeros_like(B)
    lib().shwfs_oracle_add_noise(B, B.shape[0], float(F), float(ron), int(seed), int(t), int(i), out)
    return out


def poisson_uniforms(seed, t, i, p, j=0):
    """N2: the two uniforms of pixel p of spot (t, i), attempt j."""
    u = np.zeros(2, dtype=np.float64)
    lib().shwfs_oracle_poisson_uniforms(int(seed), int(t), int(i), int(p), int(j), u)
    return u


def poisson_inversion(lam, u1):
    """N3: (k, margin) of the sequential search on u1."""
    m = C.c_double()
    k = lib().shwfs_oracle_poisson_inversion(float(lam), float(u1), C.byref(m))
    return int(k), m.value


def poisson_draw(lam, seed, t, i, p):
    """N1 + N3/N4: (k, margin) of pixel p of spot (t, i) at rate lam."""
    m = C.c_double()
    k = lib().shwfs_oracle_poisson_draw(float(lam), int(seed), int(t), int(i), int(p), C.byref(m))
    return int(k), m.value


def add_noise_poisson(B, F, ron, seed, t, i, want_margin=False):
    """N1..N5 on a D x D binned image: Poisson counts at rate F*B plus ron * (the deviate of L5)."""
    B = _c(B, np.float64)
    out = np.zeros_like(B)
    mg = np.zeros_like(B) if want_margin else None
    lib().shwfs_oracle_add_noise_poisson(B, B.shape[0], float(F), float(ron), int(seed), int(t), int(i), out,
                                         mg.ctypes.data_as(C.c_void_p) if want_margin else None)
    return (out, mg) if want_margin else out


def measure_lgs(phase, amplitude, valid_yx, n, P, b, dx, *, weight, defocus, tilt_x=None, tilt_y=None,
                cx=0.0, cy=0.0, c_phi=1.0, tau=0.0, mode=0, kernels=None, flux=0.0, ron=0.0, seed=0,
                stage=-1, nthreads=0, photon_model=0, want_margins=False):
    """L1..L6 for every frame and valid subaperture.

    phase [T,L,N,N] fp32, or [T,N,N] shared by the L = len(weight) sub-layers.  weight, defocus [rad/m^2],
    tilt_x, tilt_y [rad/m]: per sub-layer; (cx, cy) [m] centre of the quadratic.  flux = F (<= 0: no noise).
    photon_model 0: Gaussian limit (L4); 1: Poisson counts + read noise (N1..N5, shwfs_oracle_poisson.c), with
    want_margins also the per-pixel decision margins [T,nsub,D,D] of the draws.
    Returns slopes [T,nsub,2] float64, or (slopes, images[T,nsub,D,D]) for stage 2 (before noise) / 3 (after).
    """
    ph = _c(phase, np.float32)
    w = _c(weight, np.float64)
    L = w.shape[0]
    shared = ph.ndim == 3
    if shared:
        T, N, _ = ph.shape
    else:
        T, L2, N, _ = ph.shape
        assert L2 == L
    am = _c(amplitude, np.float32)
    yx = _c(valid_yx, np.int32)
    nsub = yx.shape[0]
    de = _c(defocus, np.float64)
    tx = _c(tilt_x if tilt_x is not None else np.zeros(L), np.float64)
    ty = _c(tilt_y if tilt_y is not None else np.zeros(L), np.float64)
    assert de.shape == (L,) and tx.shape == (L,) and ty.shape == (L,)
    slopes = np.zeros((T, nsub, 2), dtype=np.float64)
    kptr = None
    if kernels is not None:
        kernels = _c(kernels, np.float32)
        assert kernels.shape == (nsub, P, P), kernels.shape
        kptr = kernels.ctypes.data_as(C.c_void_p)
    images, iptr = None, None
    if stage >= 0:
        D = P // b
        images = np.zeros((T, nsub, D, D), dtype=np.float64)
        iptr = images.ctypes.data_as(C.c_void_p)
    margins = np.ones((T, nsub, P // b, P // b), dtype=np.float64) if want_margins else None
    rc = lib().shwfs_oracle_measure_lgs(ph, T, L, int(shared), N, n, P, b, am, yx, nsub, float(c_phi), float(dx),
                                        w, de, tx, ty, float(cx), float(cy), float(tau), int(mode), kptr,
                                        float(flux), float(ron), int(seed), slopes, int(stage), iptr,
                                        int(nthreads), int(photon_model),
                                        margins.ctypes.data_as(C.c_void_p) if want_margins else None)
    if rc:
        raise RuntimeError(f"shwfs_oracle_measure_lgs failed with code {rc}")
    out = (slopes, images) if stage >= 0 else slopes
    if want_margins:
        return (*out, margins) if stage >= 0 else (out, margins)
    return out

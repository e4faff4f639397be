"""Thin ctypes binding of the C-ABI library (include/shwfs.h -> paper_1408_0698_b200/libshwfs.so).

Argument marshalling only: every step of the Shack-Hartmann path runs in the CUDA kernels
behind `shwfs_measure`.  torch is used for device memory and streams and for nothing else.  There is no
CPU fallback: if the library is missing or no CUDA device is present the calls raise.

Two layers with the C names:
  * module functions `shwfs_create`, `shwfs_measure`, `shwfs_measure_host`, `shwfs_destroy`,
    `shwfs_debug_spots`, ... taking/returning raw handles and pointers (ints);
  * class `Shwfs`, the same calls on numpy / torch arrays.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libshwfs.so"

SHWFS_OK, SHWFS_EINVAL, SHWFS_EUNSUPPORTED, SHWFS_ENOMEM, SHWFS_ECUDA = 0, -1, -2, -3, -4
ALGO_AUTO, ALGO_LITERAL, ALGO_WK, ALGO_WK_GENERIC, ALGO_PRUNED_FFT, ALGO_WK_FFT = 0, 1, 2, 3, 4, 5

EXPORTS = ["shwfs_create", "shwfs_measure", "shwfs_measure_host", "shwfs_destroy", "shwfs_num_subaps",
           "shwfs_valid_list", "shwfs_pixel_scale", "shwfs_set_algorithm", "shwfs_get_algorithm",
           "shwfs_launch_count", "shwfs_debug_spots", "shwfs_strerror", "shwfs_last_cuda_error",
           "shwfs_version", "shwfs_set_sodium", "shwfs_set_noise", "shwfs_set_dm",
           "shwfs_measure_residual", "shwfs_reconstruct", "shwfs_closed_loop", "shwfs_host_bytes_per_frame",
           "shwfs_measure_host_async", "shwfs_host_wait", "shwfs_last_kernel"]
SHWFS_MAX_LAYERS = 8


class ShwfsGeometry(C.Structure):
    """struct shwfs_geometry of include/shwfs.h (field order and types must match)."""
    _fields_ = [("n_pupil", C.c_int32), ("n_sub_side", C.c_int32), ("n_pix", C.c_int32),
                ("pixel_size_m", C.c_float), ("amplitude", C.POINTER(C.c_float)), ("min_illum", C.c_float),
                ("valid_yx", C.POINTER(C.c_int32)), ("n_valid", C.c_int32), ("threshold_frac", C.c_float),
                ("threshold_mode", C.c_int32), ("phase_to_rad", C.c_float)]


class ShwfsSodium(C.Structure):
    """struct shwfs_sodium of include/shwfs.h."""
    _fields_ = [("n_layers", C.c_int32), ("shared_phase", C.c_int32), ("weight", C.POINTER(C.c_float)),
                ("defocus", C.POINTER(C.c_float)), ("tilt_x", C.POINTER(C.c_float)),
                ("tilt_y", C.POINTER(C.c_float)), ("centre_x_m", C.c_float), ("centre_y_m", C.c_float)]


class ShwfsNoise(C.Structure):
    """struct shwfs_noise of include/shwfs.h."""
    _fields_ = [("flux", C.c_float), ("read_noise", C.c_float), ("seed", C.c_uint64), ("first_frame", C.c_uint32),
                ("photon_model", C.c_int32)]


class ShwfsError(RuntimeError):
    def __init__(self, code: int, what: str):
        self.code = code
        super().__init__(what)


_lib = None


def load():
    """dlopen libshwfs.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1408_0698_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(str(LIB_PATH))
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    L.shwfs_create.argtypes = [C.POINTER(ShwfsGeometry), C.c_float, i32, i32, vp, C.POINTER(vp)]
    L.shwfs_measure.argtypes = [vp, vp, i32, vp, vp]
    L.shwfs_measure_host.argtypes = [vp, vp, i32, vp]
    L.shwfs_destroy.argtypes = [vp]
    L.shwfs_num_subaps.argtypes = [vp, C.POINTER(i32)]
    L.shwfs_valid_list.argtypes = [vp, vp]
    L.shwfs_pixel_scale.argtypes = [vp, C.POINTER(C.c_double)]
    L.shwfs_set_algorithm.argtypes = [vp, i32]
    L.shwfs_get_algorithm.argtypes = [vp, C.POINTER(i32)]
    L.shwfs_launch_count.argtypes = [vp, C.POINTER(i64)]
    L.shwfs_last_kernel.argtypes = [vp, C.c_char_p, i32]
    L.shwfs_debug_spots.argtypes = [vp, vp, i32, i32, vp, vp]
    L.shwfs_strerror.argtypes = [C.c_int]
    L.shwfs_strerror.restype = C.c_char_p
    L.shwfs_last_cuda_error.argtypes = []
    L.shwfs_last_cuda_error.restype = C.c_char_p
    L.shwfs_version.argtypes = []
    L.shwfs_set_sodium.argtypes = [vp, C.POINTER(ShwfsSodium)]
    L.shwfs_set_noise.argtypes = [vp, C.POINTER(ShwfsNoise)]
    L.shwfs_set_dm.argtypes = [vp, vp, i32]
    L.shwfs_host_bytes_per_frame.argtypes = [vp, C.POINTER(i64)]
    L.shwfs_measure_host_async.argtypes = [vp, vp, i32, vp]
    L.shwfs_host_wait.argtypes = [vp]
    L.shwfs_measure_residual.argtypes = [vp, vp, vp, i32, vp, vp]
    L.shwfs_reconstruct.argtypes = [vp, vp, vp, i32, C.c_float, vp, vp]
    L.shwfs_closed_loop.argtypes = [vp, vp, vp, C.c_float, vp, i32, vp, vp, vp]
    for name in EXPORTS:
        if name not in ("shwfs_strerror", "shwfs_last_cuda_error"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def _check(rc: int, what: str):
    if rc != SHWFS_OK:
        L = load()
        msg = L.shwfs_strerror(rc).decode()
        if rc == SHWFS_ECUDA or rc == SHWFS_ENOMEM:
            msg += " [" + L.shwfs_last_cuda_error().decode() + "]"
        raise ShwfsError(rc, f"{what}: {msg} ({rc})")


# ---- the C calls, same names, raw pointers -------------------------------------------------------

def shwfs_create(geometry: ShwfsGeometry, lambda_m: float, pad: int, bin: int, elong_kernels_ptr=None) -> int:
    out = C.c_void_p()
    _check(load().shwfs_create(C.byref(geometry), lambda_m, pad, bin, elong_kernels_ptr, C.byref(out)), "shwfs_create")
    return out.value


def shwfs_measure(handle: int, phase_dev_ptr: int, T: int, slopes_dev_ptr: int, cuda_stream: int = 0):
    _check(load().shwfs_measure(handle, phase_dev_ptr, T, slopes_dev_ptr, cuda_stream), "shwfs_measure")


def shwfs_measure_host(handle: int, phase_host_ptr: int, T: int, slopes_host_ptr: int):
    _check(load().shwfs_measure_host(handle, phase_host_ptr, T, slopes_host_ptr), "shwfs_measure_host")


def shwfs_debug_spots(handle: int, phase_dev_ptr: int, T: int, stage: int, out_dev_ptr: int, cuda_stream: int = 0):
    _check(load().shwfs_debug_spots(handle, phase_dev_ptr, T, stage, out_dev_ptr, cuda_stream), "shwfs_debug_spots")


def shwfs_destroy(handle):
    _check(load().shwfs_destroy(handle), "shwfs_destroy")


# ---- array-level convenience ---------------------------------------------------------------------

class Shwfs:
    """One wavefront sensor (one handle).  See include/shwfs.h for the meaning of every argument."""

    def __init__(self, amplitude, n_sub_side: int, n_pix: int, pixel_size_m: float, lambda_m: float, pad: int,
                 bin: int, *, min_illum: float = 0.5, valid_yx=None, threshold_frac: float = 0.0,
                 threshold_mode: int = 0, phase_to_rad: float = 1.0, elong_kernels=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1408_0698_b200 needs a CUDA device (no CPU fallback)")
        torch.cuda.init()
        torch.empty(1, device="cuda")          # make sure the primary context exists and is current
        amp = np.ascontiguousarray(amplitude, dtype=np.float32)
        if amp.ndim != 2 or amp.shape[0] != amp.shape[1]:
            raise ValueError("amplitude must be [N,N]")
        g = ShwfsGeometry()
        g.n_pupil, g.n_sub_side, g.n_pix = amp.shape[0], n_sub_side, n_pix
        g.pixel_size_m = pixel_size_m
        g.amplitude = amp.ctypes.data_as(C.POINTER(C.c_float))
        g.min_illum = min_illum
        vy = None
        if valid_yx is not None:
            vy = np.ascontiguousarray(valid_yx, dtype=np.int32).reshape(-1, 2)
            g.valid_yx = vy.ctypes.data_as(C.POINTER(C.c_int32))
            g.n_valid = vy.shape[0]
        g.threshold_frac, g.threshold_mode, g.phase_to_rad = threshold_frac, threshold_mode, phase_to_rad
        kptr = None
        if elong_kernels is not None:
            if hasattr(elong_kernels, "detach"):
                elong_kernels = elong_kernels.detach().cpu().numpy()
            k = np.ascontiguousarray(elong_kernels, dtype=np.float32)
            if k.ndim != 3 or k.shape[1] != pad or k.shape[2] != pad:
                raise ValueError("elong_kernels must be [nsub,P,P]")
            if vy is not None and k.shape[0] != vy.shape[0]:
                raise ValueError("elong_kernels and valid_yx disagree on nsub")
            if vy is None and amp.shape[0] == n_sub_side * n_pix:
                # the library reads nsub * P * P floats from this buffer before it can report nsub: count the valid
                # subapertures of the rule (include/shwfs.h: mean amplitude of the patch >= min_illum, in double)
                # first, so that too few kernels raise here instead of being read past their end
                lit = amp.astype(np.float64).reshape(n_sub_side, n_pix, n_sub_side, n_pix).sum(axis=(1, 3))
                expect = int((lit / (n_pix * n_pix) >= np.float64(np.float32(min_illum))).sum())
                if k.shape[0] != expect:
                    raise ValueError(f"elong_kernels has {k.shape[0]} entries, the valid list {expect}")
            kptr = k.ctypes.data_as(C.c_void_p)
        self._h = None
        self._h = shwfs_create(g, lambda_m, pad, bin, kptr)
        self.N, self.S, self.n, self.P, self.b, self.D = amp.shape[0], n_sub_side, n_pix, pad, bin, pad // bin
        ns = C.c_int32()
        _check(load().shwfs_num_subaps(self._h, C.byref(ns)), "shwfs_num_subaps")
        self.nsub = ns.value
        if elong_kernels is not None and k.shape[0] != self.nsub:
            self.close()
            raise ValueError(f"elong_kernels has {k.shape[0]} entries, the valid list {self.nsub}")

    # -- queries
    @property
    def valid_yx(self) -> np.ndarray:
        out = np.zeros((self.nsub, 2), dtype=np.int32)
        _check(load().shwfs_valid_list(self._h, out.ctypes.data_as(C.c_void_p)), "shwfs_valid_list")
        return out

    @property
    def pixel_scale(self) -> float:
        v = C.c_double()
        _check(load().shwfs_pixel_scale(self._h, C.byref(v)), "shwfs_pixel_scale")
        return v.value

    @property
    def algorithm(self) -> int:
        v = C.c_int32()
        _check(load().shwfs_get_algorithm(self._h, C.byref(v)), "shwfs_get_algorithm")
        return v.value

    @algorithm.setter
    def algorithm(self, algo: int):
        _check(load().shwfs_set_algorithm(self._h, int(algo)), "shwfs_set_algorithm")

    @property
    def launch_count(self) -> int:
        v = C.c_int64()
        _check(load().shwfs_launch_count(self._h, C.byref(v)), "shwfs_launch_count")
        return v.value

    @property
    def last_kernel(self) -> str:
        """Name of the kernel instance the most recent measurement launched (shwfs_last_kernel)."""
        buf = C.create_string_buffer(96)
        _check(load().shwfs_last_kernel(self._h, buf, 96), "shwfs_last_kernel")
        return buf.value.decode()

    @property
    def host_bytes_per_frame(self) -> int:
        """Bytes of one wavefront that measure_host moves over the bus (valid column runs only)."""
        v = C.c_int64()
        _check(load().shwfs_host_bytes_per_frame(self._h, C.byref(v)), "shwfs_host_bytes_per_frame")
        return v.value

    # -- the paper's full LGS model (include/shwfs.h: shwfs_set_sodium, shwfs_set_noise)
    def set_sodium(self, weight=None, defocus=None, tilt_x=None, tilt_y=None, centre=(0.0, 0.0),
                   shared_phase: bool = False):
        """Sodium sub-layers: weight[L], defocus[L] rad/m^2, tilt_x/tilt_y[L] rad/m, centre (x,y) in metres.
        weight=None returns to the single-layer sensor.  With shared_phase=False, measure() takes
        phase [T,L,N,N]."""
        if weight is None:
            _check(load().shwfs_set_sodium(self._h, None), "shwfs_set_sodium")
            self._layers = 1
            return
        f = lambda a: np.ascontiguousarray(a, dtype=np.float32)
        w, d = f(weight), f(defocus)
        sd = ShwfsSodium()
        sd.n_layers, sd.shared_phase = w.shape[0], int(bool(shared_phase))
        fp = C.POINTER(C.c_float)
        sd.weight, sd.defocus = w.ctypes.data_as(fp), d.ctypes.data_as(fp)
        keep = [w, d]
        for name, arr in (("tilt_x", tilt_x), ("tilt_y", tilt_y)):
            if arr is not None:
                a = f(arr)
                keep.append(a)
                setattr(sd, name, a.ctypes.data_as(fp))
        if d.shape != w.shape or any(a.shape != w.shape for a in keep):
            raise ValueError("weight, defocus, tilt_x, tilt_y must have the same length L")
        sd.centre_x_m, sd.centre_y_m = float(centre[0]), float(centre[1])
        _check(load().shwfs_set_sodium(self._h, C.byref(sd)), "shwfs_set_sodium")
        self._layers = 1 if shared_phase else int(w.shape[0])

    def set_noise(self, flux: float = 0.0, read_noise: float = 0.0, seed: int = 0, first_frame: int = 0,
                  photon_model: int = 0):
        """Detector noise before the centroid (flux <= 0 switches it off).  photon_model 0: Gaussian limit of the
        photon noise, 1: Poisson counts (include/shwfs.h)."""
        nz = ShwfsNoise(float(flux), float(read_noise), int(seed), int(first_frame), int(photon_model))
        _check(load().shwfs_set_noise(self._h, C.byref(nz)), "shwfs_set_noise")

    # -- closed-loop neighbours (include/shwfs.h: shwfs_set_dm, shwfs_measure_residual, shwfs_reconstruct,
    #    shwfs_closed_loop)
    def set_dm(self, modes):
        """modes: CUDA float32 [M,N,N] (None drops the DM).  The library keeps its own re-layout."""
        if modes is None:
            _check(load().shwfs_set_dm(self._h, None, 0), "shwfs_set_dm")
            self.M = 0
            return
        self._f32_cuda(modes, (None, self.N, self.N), "modes")
        _check(load().shwfs_set_dm(self._h, modes.data_ptr(), int(modes.shape[0])), "shwfs_set_dm")
        self.M = int(modes.shape[0])

    @staticmethod
    def _f32_cuda(x, shape, name):
        import torch
        ok = isinstance(x, torch.Tensor) and x.is_cuda and x.dtype == torch.float32 and x.is_contiguous() \
            and x.dim() == len(shape) and all(s is None or s == d for s, d in zip(shape, x.shape))
        if not ok:
            raise ValueError(f"{name} must be a contiguous float32 CUDA tensor of shape {shape}")

    def _stream(self, stream, like):
        import torch
        return (stream if stream is not None else torch.cuda.current_stream(like.device)).cuda_stream

    def measure_residual(self, phase, coef, out=None, stream=None):
        """Slopes of phase[t] - sum_m coef[t,m] modes[m]; coef CUDA float32 [T,M]."""
        import torch
        self._check_phase(phase)
        T = phase.shape[0]
        self._f32_cuda(coef, (T, self.M), "coef")
        if out is None:
            out = torch.empty((T, self.nsub, 2), dtype=torch.float32, device=phase.device)
        _check(load().shwfs_measure_residual(self._h, phase.data_ptr(), coef.data_ptr(), T, out.data_ptr(),
                                             self._stream(stream, phase)), "shwfs_measure_residual")
        return out

    def reconstruct(self, R, slopes, coef, gain: float = 1.0, stream=None):
        """coef[t,m] += gain * sum_k R[m,k] slopes[t,k] in place; R CUDA float32 [M, 2*nsub]."""
        T = slopes.shape[0]
        self._f32_cuda(R, (self.M, 2 * self.nsub), "R")
        self._f32_cuda(slopes, (T, self.nsub, 2), "slopes")
        self._f32_cuda(coef, (T, self.M), "coef")
        _check(load().shwfs_reconstruct(self._h, R.data_ptr(), slopes.data_ptr(), T, float(gain), coef.data_ptr(),
                                        self._stream(stream, slopes)), "shwfs_reconstruct")
        return coef

    def closed_loop(self, phase, R, gain: float, coef, want_history: bool = True, stream=None):
        """T sequential pure-integrator frames.  coef CUDA float32 [M] is c_0 on entry and c_T on return.
        Returns (slopes [T,nsub,2], hist [T,M] or None) with hist[t] = c_t."""
        import torch
        self._check_phase(phase)
        T = phase.shape[0]
        self._f32_cuda(R, (self.M, 2 * self.nsub), "R")
        self._f32_cuda(coef, (self.M,), "coef")
        slopes = torch.empty((T, self.nsub, 2), dtype=torch.float32, device=phase.device)
        hist = torch.empty((T, self.M), dtype=torch.float32, device=phase.device) if want_history else None
        _check(load().shwfs_closed_loop(self._h, phase.data_ptr(), R.data_ptr(), float(gain), coef.data_ptr(), T,
                                        slopes.data_ptr(), hist.data_ptr() if want_history else None,
                                        self._stream(stream, phase)), "shwfs_closed_loop")
        return slopes, hist

    # -- the hot path
    def _check_phase(self, phase):
        import torch
        L = getattr(self, "_layers", 1)
        shape = (self.N, self.N) if L == 1 else (L, self.N, self.N)
        ok_shape = tuple(phase.shape[1:]) == shape or (L == 1 and tuple(phase.shape[1:]) == (1, self.N, self.N))
        if not (isinstance(phase, torch.Tensor) and phase.is_cuda and phase.dtype == torch.float32
                and phase.is_contiguous() and ok_shape):
            raise ValueError(f"phase must be a contiguous float32 CUDA tensor [T,{','.join(map(str, shape))}]")

    def measure(self, phase, out=None, stream=None):
        """phase: CUDA float32 [T,N,N] -> slopes CUDA float32 [T,nsub,2] (enqueued on `stream`)."""
        import torch
        self._check_phase(phase)
        T = phase.shape[0]
        if out is None:
            out = torch.empty((T, self.nsub, 2), dtype=torch.float32, device=phase.device)
        elif not (out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and out.numel() == T * self.nsub * 2):
            raise ValueError("out must be a contiguous float32 CUDA tensor [T,nsub,2]")
        st = (stream if stream is not None else torch.cuda.current_stream(phase.device)).cuda_stream
        shwfs_measure(self._h, phase.data_ptr(), T, out.data_ptr(), st)
        return out

    def measure_host(self, phase_host, out=None):
        """phase_host: numpy or CPU torch float32 [T,N,N] -> slopes (same kind) [T,nsub,2]; synchronous."""
        is_torch = hasattr(phase_host, "data_ptr")
        if is_torch:
            if phase_host.is_cuda or not phase_host.is_contiguous() or phase_host.dtype.__str__() != "torch.float32":
                raise ValueError("phase_host must be a contiguous float32 CPU tensor")
            T, ptr = phase_host.shape[0], phase_host.data_ptr()
            if out is None:
                import torch
                out = torch.empty((T, self.nsub, 2), dtype=torch.float32, pin_memory=phase_host.is_pinned())
            optr = out.data_ptr()
        else:
            phase_host = np.ascontiguousarray(phase_host, dtype=np.float32)
            T, ptr = phase_host.shape[0], phase_host.ctypes.data
            if out is None:
                out = np.empty((T, self.nsub, 2), dtype=np.float32)
            optr = out.ctypes.data
        L = getattr(self, "_layers", 1)
        shape = (self.N, self.N) if L == 1 else (L, self.N, self.N)
        if tuple(phase_host.shape[1:]) != shape:
            raise ValueError(f"phase_host must be [T,{','.join(map(str, shape))}]")
        shwfs_measure_host(self._h, ptr, T, optr)
        return out

    def measure_host_async(self, phase_host, out):
        """Enqueue measure_host on the handle's own streams (pinned CPU torch tensors only); host_wait() ends it."""
        if not (phase_host.is_pinned() and out.is_pinned() and phase_host.is_contiguous() and out.is_contiguous()):
            raise ValueError("measure_host_async needs contiguous pinned CPU tensors")
        _check(load().shwfs_measure_host_async(self._h, phase_host.data_ptr(), int(phase_host.shape[0]),
                                               out.data_ptr()), "shwfs_measure_host_async")
        return out

    def host_wait(self):
        _check(load().shwfs_host_wait(self._h), "shwfs_host_wait")

    def debug_spots(self, phase, stage: int, stream=None):
        """Images of stage 0 / 1 ([T,nsub,P,P]) or 2 / 3 ([T,nsub,D,D]; 3 = after the detector noise) as a
        CUDA tensor (parity only)."""
        import torch
        self._check_phase(phase)
        T = phase.shape[0]
        side = self.D if stage >= 2 else self.P
        out = torch.empty((T, self.nsub, side, side), dtype=torch.float32, device=phase.device)
        st = (stream if stream is not None else torch.cuda.current_stream(phase.device)).cuda_stream
        shwfs_debug_spots(self._h, phase.data_ptr(), T, stage, out.data_ptr(), st)
        return out

    def close(self):
        if getattr(self, "_h", None):
            shwfs_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()


def from_config(cfg, wfs: int = 0, *, kernels="auto", **overrides) -> "Shwfs":
    """Build the sensor of one workloads.WfsConfig (mask, tau and -- when the config has elongation --
    the kernels of WFS `wfs`, evaluated on the GPU by workloads.elongation_kernels)."""
    from . import workloads as W
    amp = W.pupil_mask(cfg)
    kw = dict(min_illum=cfg.min_illum, threshold_frac=cfg.tau)
    kw.update(overrides)
    k = None
    if isinstance(kernels, str) and kernels == "auto" and cfg.elong_max_arcsec > 0:
        import torch
        with Shwfs(amp, cfg.S, cfg.n, cfg.dx, W.LAMBDA_M, cfg.P, cfg.b, **kw) as probe:
            yx = probe.valid_yx            # the library's own H0 valid list (no kernels needed for it)
        k = W.elongation_kernels(cfg, wfs, yx, device=torch.device("cuda"))
        kw.setdefault("valid_yx", yx)
    elif kernels is not None and not isinstance(kernels, str):
        k = kernels
    return Shwfs(amp, cfg.S, cfg.n, cfg.dx, W.LAMBDA_M, cfg.P, cfg.b, elong_kernels=k, **kw)


# ---- pyramid wavefront sensor (include/pyrwfs.h) -------------------------------------------------------

PYR_EXPORTS = ["pyrwfs_create", "pyrwfs_destroy", "pyrwfs_num_pixels", "pyrwfs_valid_list", "pyrwfs_launch_count",
               "pyrwfs_measure", "pyrwfs_debug_quadrants"]


class PyrwfsConfig(C.Structure):
    """struct pyrwfs_config of include/pyrwfs.h (field order and types must match)."""
    _fields_ = [("n_pupil", C.c_int32), ("amplitude", C.POINTER(C.c_float)), ("min_illum", C.c_float),
                ("pad", C.c_int32), ("separation", C.c_int32), ("bin", C.c_int32), ("mod_radius", C.c_float),
                ("mod_points", C.c_int32), ("pupil_diameter_px", C.c_float), ("phase_to_rad", C.c_float)]


def _pyr_lib():
    L = load()
    if not getattr(L, "_pyr_ready", False):
        vp, i32 = C.c_void_p, C.c_int32
        L.pyrwfs_create.argtypes = [C.POINTER(PyrwfsConfig), C.POINTER(vp)]
        L.pyrwfs_destroy.argtypes = [vp]
        L.pyrwfs_num_pixels.argtypes = [vp, C.POINTER(i32)]
        L.pyrwfs_valid_list.argtypes = [vp, vp]
        L.pyrwfs_launch_count.argtypes = [vp, C.POINTER(C.c_int64)]
        L.pyrwfs_measure.argtypes = [vp, vp, i32, vp, vp]
        L.pyrwfs_debug_quadrants.argtypes = [vp, vp, i32, vp, vp]
        for name in PYR_EXPORTS:
            getattr(L, name).restype = C.c_int
        L._pyr_ready = True
    return L


class Pyrwfs:
    """One pyramid sensor (one handle).  See include/pyrwfs.h for the meaning of every argument."""

    def __init__(self, amplitude, pad: int, separation: int, bin: int, mod_radius: float, mod_points: int,
                 pupil_diameter_px: float, *, min_illum: float = 0.5, phase_to_rad: float = 1.0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1408_0698_b200 needs a CUDA device (no CPU fallback)")
        torch.empty(1, device="cuda")
        amp = np.ascontiguousarray(amplitude, dtype=np.float32)
        if amp.ndim != 2 or amp.shape[0] != amp.shape[1]:
            raise ValueError("amplitude must be [N,N]")
        cfg = PyrwfsConfig(amp.shape[0], amp.ctypes.data_as(C.POINTER(C.c_float)), min_illum, pad, separation, bin,
                           mod_radius, mod_points, pupil_diameter_px, phase_to_rad)
        out = C.c_void_p()
        self._h = None
        _check(_pyr_lib().pyrwfs_create(C.byref(cfg), C.byref(out)), "pyrwfs_create")
        self._h = out.value
        self.N, self.Np, self.s, self.bp, self.Sp = amp.shape[0], pad, separation, bin, amp.shape[0] // bin
        nv = C.c_int32()
        _check(_pyr_lib().pyrwfs_num_pixels(self._h, C.byref(nv)), "pyrwfs_num_pixels")
        self.nvalid = nv.value

    @property
    def valid_yx(self) -> np.ndarray:
        out = np.zeros((self.nvalid, 2), dtype=np.int32)
        _check(_pyr_lib().pyrwfs_valid_list(self._h, out.ctypes.data_as(C.c_void_p)), "pyrwfs_valid_list")
        return out

    @property
    def launch_count(self) -> int:
        v = C.c_int64()
        _check(_pyr_lib().pyrwfs_launch_count(self._h, C.byref(v)), "pyrwfs_launch_count")
        return v.value

    def _check_phase(self, phase):
        import torch
        if not (isinstance(phase, torch.Tensor) and phase.is_cuda and phase.dtype == torch.float32
                and phase.is_contiguous() and tuple(phase.shape[1:]) == (self.N, self.N)):
            raise ValueError(f"phase must be a contiguous float32 CUDA tensor [T,{self.N},{self.N}]")

    def measure(self, phase, out=None, stream=None):
        """phase CUDA float32 [T,N,N] -> signals CUDA float32 [T,nvalid,2]."""
        import torch
        self._check_phase(phase)
        T = phase.shape[0]
        if out is None:
            out = torch.empty((T, self.nvalid, 2), dtype=torch.float32, device=phase.device)
        st = (stream if stream is not None else torch.cuda.current_stream(phase.device)).cuda_stream
        _check(_pyr_lib().pyrwfs_measure(self._h, phase.data_ptr(), T, out.data_ptr(), st), "pyrwfs_measure")
        return out

    def debug_quadrants(self, phase, stream=None):
        """Binned quadrant images Q [T,2,2,Sp,Sp] (parity only)."""
        import torch
        self._check_phase(phase)
        T = phase.shape[0]
        out = torch.empty((T, 2, 2, self.Sp, self.Sp), dtype=torch.float32, device=phase.device)
        st = (stream if stream is not None else torch.cuda.current_stream(phase.device)).cuda_stream
        _check(_pyr_lib().pyrwfs_debug_quadrants(self._h, phase.data_ptr(), T, out.data_ptr(), st),
               "pyrwfs_debug_quadrants")
        return out

    def close(self):
        if getattr(self, "_h", None):
            _check(_pyr_lib().pyrwfs_destroy(self._h), "pyrwfs_destroy")
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

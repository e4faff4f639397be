"""Whole kernels of csrc/ on the host: each kernel is cut out of its .cu file as text, compiled by g++ with the headers
it includes as they are, and run thread by thread on the coroutine SIMT machine of tests/host/simt.h (shared memory,
shuffles, __syncwarp / __syncthreads, the chunk counter of the dynamic deal, TMA boxes with their swizzle and
mbarriers, cp.async batches) on the same seeded inputs as the float64 oracles: Shack-Hartmann kernels (pruned_fft.cu,
wk.cu, wk_fft.cu, literal.cu; the sodium / noise / DM-residual instances) binned images within 1e-4 of the spot peak
and slopes within 1e-3 px (north_star) for every spot; pyramid.cu quadrants 1e-4 of peak, signals 2e-4; loop.cu
against the definitions C1 / C2 of oracle/closed_loop.py; the operand kernels of dm_umma.cu against the plain GEMM.
Each case runs under up to three thread orders (ascending, descending, seeded random between synchronisation points)
and must give bit-identical results: a barrier the code needs and does not have shows up as a difference -- and one
mutant per kernel family, built from the same text with such a barrier removed, must fail (MUTANTS).  Whole frames at
BASELINE.json's geometry: config 3 (every spot), config 2 (every spot), config 5 (every 7th subaperture), the LBT-like
pyramid.  CPU-side parity of device code, thread mapping included: no GPU."""
import dataclasses
import re
import shutil
import struct
import subprocess
from pathlib import Path

import numpy as np
import pytest

from oracle import shwfs_oracle as O
from paper_1408_0698_b200 import workloads as W

ROOT = Path(__file__).resolve().parent.parent
CSRC = ROOT / "paper_1408_0698_b200" / "csrc"
CUDA_INC = Path("/usr/local/cuda/include")
PATCH_LIT = 1 << 30

def small_config(base: int, S: int, **kw) -> W.WfsConfig:
    """The geometry of config `base` on S x S subapertures: same n, P, b, pixel size and wavelength; the pupil radii
    scaled to the smaller grid so that fully lit, partially lit and dark subapertures all occur."""
    c = W.CONFIGS[base]
    N = S * c.n
    r_out = 0.5 * N * c.dx
    return dataclasses.replace(c, N=N, S=S, r_out=r_out, r_in=r_out * c.r_in / c.r_out if c.r_out else 0.0,
                               screen_M=256, **kw)


def cut(src: str, begin: str, end: str) -> str:
    assert src.count(begin) == 1 and src.count(end) == 1, (begin, end)
    block = src[src.index(begin):src.index(end)]
    assert "<<<" not in block
    return block


MUTANTS = {
    # the machine does see a missing barrier: each entry removes one the kernel needs
    "pf_mut": ("pf", ("__syncwarp();                                      /* rows visible; the staging slot has been read */", "")),
    "wk_mut": ("wk", ("if (pass == 1) __syncthreads();", "")),
    "wkf_mut": ("wkf", ("    }   /* sub-layers */\n    __syncwarp();", "    }   /* sub-layers */\n")),
    "lit_mut": ("lit", ("    for (int v = 0; v < P; ++v) Sh[(v ^ HP) * LD + (r ^ HP)] = re[v];\n    __syncthreads();",
                        "    for (int v = 0; v < P; ++v) Sh[(v ^ HP) * LD + (r ^ HP)] = re[v];\n")),
    "loop_mut": ("loop", ("        __syncthreads();                                    /* stage (ch & 1) is refilled two chunks later */", "")),
    "pyr_mut": ("pyr", ("    __syncwarp();\n#pragma unroll\n    for (int jj = 0; jj < R; jj += 2) {",
                        "#pragma unroll\n    for (int jj = 0; jj < R; jj += 2) {")),
}


@pytest.fixture(scope="module")
def harnesses(tmp_path_factory):
    """Every harness and every mutant, each in a directory of its own with the kernel text cut out for it, compiled
    side by side (g++ -O0 -ffp-contract=off: the fmaf calls of the shims are the only contractions)."""
    if shutil.which("g++") is None or not (CUDA_INC / "cuda_runtime.h").exists():
        pytest.skip("needs g++ and the CUDA headers")
    jobs = {}
    for key in ("pf", "wk", "lit", "pyr", "loop", *MUTANTS):
        base, mutate = MUTANTS.get(key, (key, None))
        d = tmp_path_factory.mktemp(key)
        if base == "pf":
            pf_extract(d, mutate)
        elif base == "wk":
            wk_extract(d, mutate)
        elif base == "wkf":
            wk_extract(d, None, mutate)
        elif base == "lit":
            lit_extract(d, mutate)
        elif base == "loop":
            loop_extract(d, mutate)
        else:
            pyr_extract(d, mutate)
        name = {"pf": "pf", "wk": "wk", "wkf": "wk", "lit": "lit", "pyr": "pyr", "loop": "loop"}[base] + "_kernel_harness"
        exe = d / name
        proc = subprocess.Popen(["g++", "-std=c++17", "-O0", "-ffp-contract=off", f"-I{CUDA_INC}", f"-I{d}", "-Wno-attributes",
                                 "-Wno-psabi", "-o", str(exe), str(ROOT / "tests" / "host" / f"{name}.cpp")],
                                stdout=subprocess.DEVNULL, stderr=subprocess.PIPE, text=True)
        jobs[key] = (proc, exe)
    out = {}
    for key, (proc, exe) in jobs.items():
        _, err = proc.communicate(timeout=900)
        assert proc.returncode == 0, key + ": " + err[-3000:]
        out[key] = exe
    return out


def patch_table(amp: np.ndarray, yx: np.ndarray, n: int) -> np.ndarray:
    """What shwfs_create puts into the handle (api.cu, "patch table"): origin in pixels, flag for all-ones patches."""
    out = np.zeros((len(yx), 2), np.int32)
    for i, (sy, sx) in enumerate(yx):
        lit = bool(np.all(amp[sy * n:(sy + 1) * n, sx * n:(sx + 1) * n] == 1.0))
        out[i] = (sx * n | (PATCH_LIT if lit else 0), sy * n)
    return out


def compare(got_slopes, got_img, want_slopes, want_img, tau, mode, label):
    assert not np.isnan(got_slopes).any() and not np.isnan(got_img).any(), f"{label}: a spot was never written"
    peak = want_img.max(axis=(2, 3), keepdims=True)
    ierr = float((np.abs(got_img - want_img) / peak).max())
    assert ierr <= 1e-4, (label, ierr)
    serr = np.abs(got_slopes - want_slopes).max(axis=2)
    if mode == 1:
        # hard mask: compare the spots none of whose pixels sits within rounding of the threshold (tests/test_parity_gpu.py)
        clear = (np.abs(want_img - tau * peak) > 2e-4 * peak).all(axis=(2, 3))
        assert clear.mean() > 0.5, label
        serr = serr[clear]
    assert float(serr.max()) <= 1e-3, (label, float(serr.max()))
    return ierr, float(serr.max())


# ---------------------------------------------------------------- pruned_fft_kernel (config 2's kernel)

PF_CASES = [
    # base config, S, T, mode, tau, instances [(tma, chunk, lazy)]
    (2, 6, 5, 0, 0.10, [(0, 0, 0), (1, 0, 0), (1, 4, 1), (0, 4, 0)]),     # n = 16, P = 32: <32,16>
    (1, 10, 3, 0, 0.0, [(0, 0, 0), (0, 4, 0)]),                           # config 1 itself, n = 8, P = 16: <16,8>
    (3, 8, 3, 1, 0.10, [(0, 0, 0)]),                                      # n = 10 < NZ = 16, P = 32, hard threshold
    (5, 6, 3, 0, 0.10, [(1, 4, 0), (0, 0, 0)]),                           # n = 16, P = 64, b = 4: <64,16>
]


def pf_extract(tmp_path: Path, mutate=None) -> None:
    src = (CSRC / "pruned_fft.cu").read_text()
    block = cut(src, "constexpr int PF_THREADS", "template <int P, int NZ, int MODE, bool TMA>\ncudaError_t launch_pf_inst")
    block, k = re.subn(r"extern __shared__ __align__\(16\) unsigned char pf_smem\[\];",
                       "unsigned char *pf_smem = simt::smem();", block)
    assert k == 1 and "pruned_fft_kernel(const PfArgs A" in block and "cog16<MODE>" in block
    if mutate is not None:
        assert block.count(mutate[0]) == 1, mutate[0]
        block = block.replace(mutate[0], mutate[1])
    (tmp_path / "pf_kernel_extract.inc").write_text(block)


def pf_run(exe, tmp_path, c, T, nsub, mode, tau, ph, amp, table, tma, chunk, lazy, grid, order, seed):
    """One simulated launch; returns (slopes, binned images, stdout) or None when the harness reports a failure."""
    fin, fout = tmp_path / "in.bin", tmp_path / "out.bin"
    with open(fin, "wb") as f:
        f.write(struct.pack("14i", c.N, c.n, c.P, T, nsub, mode, tma, chunk, grid, order, seed, lazy, 0, 0))
        f.write(struct.pack("2f", tau, 1.0))
        f.write(ph.astype(np.float32).tobytes())
        f.write(amp.astype(np.float32).tobytes())
        f.write(table.tobytes())
    r = subprocess.run([str(exe), str(fin), str(fout)], capture_output=True, text=True, timeout=600)
    if r.returncode != 0 or not r.stdout.startswith("ok "):
        assert r.stdout.startswith("FAIL"), r.stdout[-500:] + r.stderr[-500:]
        return None
    raw = np.fromfile(fout, np.float32)
    ns, ni = T * nsub * 2, T * nsub * 256
    got = raw[:ns].reshape(T, nsub, 2).astype(np.float64)
    img = raw[ns:ns + ni].reshape(T, nsub, 16, 16).astype(np.float64)
    counters = raw[ns + ni:].view(np.int32)
    assert (counters == 0).all(), f"chunk counters not re-armed: {counters}"
    return got, img, r.stdout


def test_pruned_fft_kernel_whole_on_the_host(tmp_path, harnesses):
    exe = harnesses["pf"]

    runs = 0
    for base, S, T, mode, tau, instances in PF_CASES:
        c = W.CONFIGS[1] if (base, S) == (1, 10) else small_config(base, S)
        amp = W.pupil_mask(c)
        yx = O.valid_list(amp, c.n, c.min_illum)
        ph = W.phase_frames(c, 0, range(T))
        nsub = len(yx)
        table = patch_table(amp, yx, c.n)
        lit = (table[:, 0] & PATCH_LIT) != 0
        if base != 1:
            assert lit.any() and (~lit).any(), "the case should have both kinds of subaperture"
        want, wimg = O.measure(ph, amp, yx, c.n, c.P, c.b, tau=tau, mode=mode, stage=2)
        for tma, chunk, lazy in instances:
            first = None
            for order, grid in ((0, 3), (1, 3), (2, 2)):
                if chunk:
                    # the launcher deals chunks only when every warp has work; keep that in the small case
                    grid = max(1, min(grid, (T * nsub) // (4 * chunk)))
                label = f"config {base} S={S} tma={tma} chunk={chunk} lazy={lazy} order={order} grid={grid}"
                out = pf_run(exe, tmp_path, c, T, nsub, mode, tau, ph, amp, table, tma, chunk, lazy, grid, order, 1408 + runs)
                assert out is not None, label
                got, img, stdout = out
                words = stdout.split()
                boxes = int(words[words.index("boxes") + 1])
                assert boxes == (T * nsub if tma else 0) and words[-1] == "0", f"{label}: {stdout}"
                compare(got, img, want, wimg, tau, mode, label)
                # same arithmetic whatever the thread order and the grid: bit-identical
                if first is None:
                    first = (got, img)
                else:
                    assert np.array_equal(first[0], got) and np.array_equal(first[1], img), f"{label}: depends on the thread order"
                runs += 1
    assert runs == 27

    # the machine does see a missing barrier: without the __syncwarp between the row pass and the column pass the
    # register-gather instance reads rows nobody has written yet (wrong images), and the TMA instance re-arms a
    # staging slot other lanes still wait for (the launch hangs)
    mutant = harnesses["pf_mut"]
    c = small_config(2, 6)
    amp = W.pupil_mask(c)
    yx = O.valid_list(amp, c.n, c.min_illum)
    ph = W.phase_frames(c, 0, range(2))
    table = patch_table(amp, yx, c.n)
    want, wimg = O.measure(ph, amp, yx, c.n, c.P, c.b, tau=0.1, stage=2)
    for tma in (0, 1):
        out = pf_run(mutant, tmp_path, c, 2, len(yx), 0, 0.1, ph, amp, table, tma, 0, 0, 2, 0, 1)
        if out is not None:
            with pytest.raises(AssertionError):
                compare(out[0], out[1], want, wimg, 0.1, 0, "mutant")


# ---------------------------------------------------------------- wk.cu: table kernel + the headline kernel

def wkf_extract(tmp_path: Path, mutate=None) -> None:
    src = (CSRC / "wk_fft.cu").read_text()
    block = cut(src, "constexpr int WF_ROWS = 16;", "template <int n, int MODE, int EXTK, bool TMA>\ncudaError_t launch_wkf_inst")
    block, k1 = re.subn(r"extern __shared__ __align__\(16\) unsigned char wf_smem\[\];", "unsigned char *wf_smem = simt::smem();", block)
    # the table row staging is inline PTX (cp.async): the harness restates its copies
    block, k2 = re.subn(r"\bmrow_stage<n>\(", "host_mrow_stage<n>(", block)
    block, k3 = re.subn(r"\bmrow_wait\(\)", "host_mrow_wait()", block)
    assert (k1, k2, k3) == (1, 1, 1) and "wkf_kernel(const WkArgs A" in block
    if mutate is not None:
        assert block.count(mutate[0]) == 1, mutate[0]
        block = block.replace(mutate[0], mutate[1])
    (tmp_path / "wkf_kernel_extract.inc").write_text(block)


def wk_extract(tmp_path: Path, mutate=None, mutate_fft=None) -> None:
    src = (CSRC / "wk.cu").read_text()
    block = cut(src, "__global__ void wk_table_kernel(", "template <int n, int MODE, int EXTK>\ncudaError_t launch_special_mode")
    block, k1 = re.subn(r"extern __shared__ double2 tmp\[\];", "double2 *tmp = reinterpret_cast<double2 *>(simt::smem());", block)
    block, k2 = re.subn(r"extern __shared__ __align__\(16\) float smem\[\];",
                        "float *smem = reinterpret_cast<float *>(simt::smem());", block)
    assert (k1, k2) == (1, 2) and "wk_measure_kernel(const WkArgs A)" in block and "wk_generic_kernel(const WkArgs A" in block
    if mutate is not None:
        assert block.count(mutate[0]) == 1, mutate[0]
        block = block.replace(mutate[0], mutate[1])
    (tmp_path / "wk_kernel_extract.inc").write_text(block)
    wkf_extract(tmp_path, mutate_fft)


def wk_run(exe, tmp_path, c, T, yx, mode, tau, ph, amp, K, kernel, order, seed, L=0, sod_q=(), sod_sw=(), sod_g=None,
           grid=0, lazy=0, shared=1, flux=0.0, ron=0.0, noise_seed=0, photon_model=0, dm_patch=None):
    """kernel: 0 wk_measure_kernel, 1 wk_generic_kernel, 2 wkf_kernel one tile per CTA, 3 wkf_kernel persistent (TMA)."""
    nsub = len(yx)
    fin, fout = tmp_path / "in.bin", tmp_path / "out.bin"
    with open(fin, "wb") as f:
        f.write(struct.pack("14i", c.N, c.n, c.P, c.b, T, nsub, mode, int(K is not None), kernel, order, seed, L, grid, lazy))
        f.write(struct.pack("2f", tau, 1.0))
        f.write(np.resize(np.asarray(list(sod_q) + [0.0] * 8, np.float32), 8).tobytes())
        f.write(np.resize(np.asarray(list(sod_sw) + [0.0] * 8, np.float32), 8).tobytes())
        f.write(struct.pack("2f2i2Ii", flux, ron, shared, photon_model, noise_seed & 0xffffffff, noise_seed >> 32,
                            int(dm_patch is not None)))
        f.write(np.ascontiguousarray(ph, np.float32).tobytes())
        f.write(np.ascontiguousarray(amp, np.float32).tobytes())
        f.write(np.ascontiguousarray(yx, np.int32).tobytes())
        if K is not None:
            f.write(np.ascontiguousarray(K, np.float32).tobytes())
        if sod_g is not None:
            f.write(np.ascontiguousarray(sod_g, np.float32).tobytes())
        if dm_patch is not None:
            f.write(np.ascontiguousarray(dm_patch, np.float32).tobytes())
    r = subprocess.run([str(exe), str(fin), str(fout)], capture_output=True, text=True, timeout=900)
    if r.returncode != 0 or not r.stdout.startswith("ok "):
        assert r.stdout.startswith("FAIL"), r.stdout[-500:] + r.stderr[-500:]
        return None
    raw = np.fromfile(fout, np.float32)
    D = c.P // c.b
    ns, ni = T * nsub * 2, T * nsub * D * D
    out = (raw[:ns].reshape(T, nsub, 2).astype(np.float64), raw[ns:ns + ni].reshape(T, nsub, D, D).astype(np.float64))
    if flux > 0:
        out += (raw[ns + ni:].reshape(T, nsub, D, D).astype(np.float64),)
    return out


WK_CASES = [
    # base config, S, T, mode, tau, elongation kernels, generic kernel too
    (3, 8, 3, 0, 0.10, True, True),       # n = 10, P = 32, b = 2 with per-subaperture kernels: the headline instance
    (3, 8, 1, 1, 0.10, False, False),     # the same without kernels (shared table), hard threshold
    (1, 10, 3, 0, 0.0, False, True),      # config 1 itself: n = 8, P = 16, b = 1
    (5, 6, 2, 0, 0.10, True, False),      # n = 16, P = 64, b = 4 with kernels
]


def test_lag_domain_kernels_whole_on_the_host(tmp_path, harnesses):
    exe = harnesses["wk"]
    runs = 0
    for base, S, T, mode, tau, with_k, generic_too in WK_CASES:
        c = W.CONFIGS[1] if (base, S) == (1, 10) else small_config(base, S)
        amp = W.pupil_mask(c)
        yx = O.valid_list(amp, c.n, c.min_illum)
        ph = W.phase_frames(c, 0, range(T))
        K = W.elongation_kernels(c, 0, yx) if with_k else None
        assert (T * len(yx)) % 32 != 0, "the last CTA should be ragged"
        want, wimg = O.measure(ph, amp, yx, c.n, c.P, c.b, tau=tau, mode=mode, kernels=K, stage=2)
        first = None
        for order in (0, 1, 2):
            label = f"config {base} S={S} kernels={with_k} order={order}"
            out = wk_run(exe, tmp_path, c, T, yx, mode, tau, ph, amp, K, 0, order, 698 + runs)
            assert out is not None, label
            compare(out[0], out[1], want, wimg, tau, mode, label)
            if first is None:
                first = out
            else:
                assert np.array_equal(first[0], out[0]) and np.array_equal(first[1], out[1]), f"{label}: depends on the thread order"
            runs += 1
        if with_k and c.n == 10:
            # the headline instance under five more random interleavings of its 160-thread CTAs
            for seed in range(5):
                out = wk_run(exe, tmp_path, c, T, yx, mode, tau, ph, amp, K, 0, 2, 9000 + seed)
                assert out is not None and np.array_equal(first[0], out[0]) and np.array_equal(first[1], out[1]), seed
        if generic_too and mode == 0:
            # the size-generic kernel: one frame, an independently written cross-check of the same table
            out = wk_run(exe, tmp_path, c, 1, yx, mode, tau, ph[:1], amp, K, 1, 2, 5)
            assert out is not None
            compare(out[0], out[1], want[:1], wimg[:1], tau, mode, f"config {base} generic")
            runs += 1
    assert runs == 14

    # the barrier the round-1 review worried about: the second-pass rows of H overwrite the field buffer "behind one
    # __syncthreads()" -- without it a warp that finishes its lag row early destroys field rows other warps still
    # read, and the machine shows it (wrong images under at least one thread order)
    mutant = harnesses["wk_mut"]
    c = small_config(3, 8)
    amp = W.pupil_mask(c)
    yx = O.valid_list(amp, c.n, c.min_illum)
    ph = W.phase_frames(c, 0, range(1))
    want, wimg = O.measure(ph, amp, yx, c.n, c.P, c.b, tau=0.1, stage=2)
    caught = 0
    for order in (0, 1, 2):
        out = wk_run(mutant, tmp_path, c, 1, yx, 0, 0.1, ph, amp, None, 0, order, 9)
        try:
            assert out is not None
            compare(out[0], out[1], want, wimg, 0.1, 0, "mutant")
        except AssertionError:
            caught += 1
    assert caught >= 1


# ---------------------------------------------------------------- wk_fft.cu: autocorrelation by FFT (config 5's kernel)

WKF_CASES = [
    # base config, S, T, mode, tau, elongation kernels, n override, instances [(kernel, grid, lazy)]
    (5, 6, 5, 0, 0.10, True, None, [(2, 0, 0), (3, 2, 0), (3, 3, 1)]),    # n = 16, P = 64, b = 4: ldg, persistent TMA
    (3, 8, 2, 0, 0.10, True, None, [(2, 0, 0)]),                          # n = 10: what AUTO gives a two-frame call
    (1, 10, 1, 1, 0.05, False, None, [(2, 0, 0)]),                        # config 1 itself, n = 8, hard threshold
    (5, 6, 1, 0, 0.10, True, 12, [(2, 0, 0)]),                            # n = 12 (threads r >= n idle), P = 64
    (2, 6, 1, 0, 0.10, False, 14, [(2, 0, 0)]),                           # n = 14, P = 32, shared table
]


def test_fft_autocorrelation_kernel_whole_on_the_host(tmp_path, harnesses):
    exe = harnesses["wk"]
    runs = 0
    for base, S, T, mode, tau, with_k, n_over, instances in WKF_CASES:
        c = W.CONFIGS[1] if (base, S) == (1, 10) else small_config(base, S)
        if n_over is not None:
            c = dataclasses.replace(c, n=n_over, N=S * n_over, r_out=0.5 * S * n_over * c.dx,
                                    r_in=0.5 * S * n_over * c.dx * W.CONFIGS[base].r_in / W.CONFIGS[base].r_out)
        amp = W.pupil_mask(c)
        yx = O.valid_list(amp, c.n, c.min_illum)
        ph = W.phase_frames(c, 0, range(T))
        K = W.elongation_kernels(c, 0, yx) if with_k else None
        want, wimg = O.measure(ph, amp, yx, c.n, c.P, c.b, tau=tau, mode=mode, kernels=K, stage=2)
        for kernel, grid, lazy in instances:
            first = None
            for order in (0, 1, 2):
                label = f"config {base} S={S} n={c.n} kernel={kernel} grid={grid} lazy={lazy} order={order}"
                out = wk_run(exe, tmp_path, c, T, yx, mode, tau, ph, amp, K, kernel, order, 55 + runs, grid=grid, lazy=lazy)
                assert out is not None, label
                compare(out[0], out[1], want, wimg, tau, mode, label)
                if first is None:
                    first = out
                else:
                    assert np.array_equal(first[0], out[0]) and np.array_equal(first[1], out[1]), f"{label}: depends on the thread order"
                runs += 1
    assert runs == 21

    # a missing __syncwarp between step C (every thread writes its two columns of g) and step D (a thread reads a row)
    mutant = harnesses["wkf_mut"]
    c = small_config(5, 6)
    amp = W.pupil_mask(c)
    yx = O.valid_list(amp, c.n, c.min_illum)
    ph = W.phase_frames(c, 0, range(1))
    want, wimg = O.measure(ph, amp, yx, c.n, c.P, c.b, tau=0.1, stage=2)
    caught = 0
    for order in (0, 1, 2):
        out = wk_run(mutant, tmp_path, c, 1, yx, 0, 0.1, ph, amp, None, 2, order, 9)
        try:
            assert out is not None
            compare(out[0], out[1], want, wimg, 0.1, 0, "mutant")
        except AssertionError:
            caught += 1
    assert caught >= 1


# ---------------------------------------------------------------- literal.cu: the chain as the paper words it

def lit_extract(tmp_path: Path, mutate=None) -> None:
    src = (CSRC / "literal.cu").read_text()
    block = cut(src, "constexpr int LIT_THREADS = 128;", "template <int P, int NZ>\ncudaError_t launch_literal")
    block, k1 = re.subn(r"extern __shared__ __align__\(16\) float2 lit_smem\[\];",
                        "float2 *lit_smem = reinterpret_cast<float2 *>(simt::smem());", block)
    block, k2 = re.subn(r"extern __shared__ double2 ksm\[\];", "double2 *ksm = reinterpret_cast<double2 *>(simt::smem());", block)
    assert (k1, k2) == (1, 1) and "literal_kernel(const LitArgs A)" in block and "literal_khat_kernel(" in block
    if mutate is not None:
        assert block.count(mutate[0]) == 1, mutate[0]
        block = block.replace(mutate[0], mutate[1])
    (tmp_path / "lit_kernel_extract.inc").write_text(block)


def lit_run(exe, tmp_path, c, T, yx, mode, tau, ph, amp, K, stage, order, seed):
    nsub = len(yx)
    fin, fout = tmp_path / "in.bin", tmp_path / "out.bin"
    with open(fin, "wb") as f:
        f.write(struct.pack("12i", c.N, c.n, c.P, c.b, T, nsub, mode, int(K is not None), stage, order, seed, 0))
        f.write(struct.pack("2f", tau, 1.0))
        f.write(np.ascontiguousarray(ph, np.float32).tobytes())
        f.write(np.ascontiguousarray(amp, np.float32).tobytes())
        f.write(np.ascontiguousarray(yx, np.int32).tobytes())
        if K is not None:
            f.write(np.ascontiguousarray(K, np.float32).tobytes())
    r = subprocess.run([str(exe), str(fin), str(fout)], capture_output=True, text=True, timeout=900)
    if r.returncode != 0 or not r.stdout.startswith("ok "):
        assert r.stdout.startswith("FAIL"), r.stdout[-500:] + r.stderr[-500:]
        return None
    raw = np.fromfile(fout, np.float32)
    side = c.P // c.b if stage == 2 else c.P
    ns = T * nsub * 2
    return raw[:ns].reshape(T, nsub, 2).astype(np.float64), raw[ns:].reshape(T, nsub, side, side).astype(np.float64)


LIT_CASES = [
    # base config, S, T, mode, tau, elongation kernels, stages
    (3, 8, 2, 0, 0.10, True, (2, 1)),     # n = 10, P = 32 <32,32>: binned image and the convolved image before binning
    (2, 6, 1, 1, 0.10, False, (2, 0)),    # n = 16, P = 32 <32,16>: no kernels, hard threshold; stage 0 = intensity
    (1, 10, 3, 0, 0.0, False, (2,)),      # config 1 itself: P = 16 <16,8>, two spots per warp
    (5, 4, 1, 0, 0.10, True, (2,)),       # P = 64 <64,32>: two warps per spot, reductions through shared memory
]


def test_literal_chain_kernels_whole_on_the_host(tmp_path, harnesses):
    exe = harnesses["lit"]
    runs = 0
    for base, S, T, mode, tau, with_k, stages in LIT_CASES:
        c = W.CONFIGS[1] if (base, S) == (1, 10) else small_config(base, S)
        amp = W.pupil_mask(c)
        yx = O.valid_list(amp, c.n, c.min_illum)
        ph = W.phase_frames(c, 0, range(T))
        K = W.elongation_kernels(c, 0, yx) if with_k else None
        for stage in stages:
            want, wimg = O.measure(ph, amp, yx, c.n, c.P, c.b, tau=tau, mode=mode, kernels=K, stage=stage)
            first = None
            for order in (0, 1, 2):
                label = f"config {base} S={S} stage={stage} order={order}"
                out = lit_run(exe, tmp_path, c, T, yx, mode, tau, ph, amp, K, stage, order, 77 + runs)
                assert out is not None, label
                if stage == 2:
                    compare(out[0], out[1], want, wimg, tau, mode, label)
                else:
                    peak = wimg.max(axis=(2, 3), keepdims=True)
                    assert float((np.abs(out[1] - wimg) / peak).max()) <= 1e-4, label
                if first is None:
                    first = out
                else:
                    assert np.array_equal(first[0], out[0]) and np.array_equal(first[1], out[1]), f"{label}: depends on the thread order"
                runs += 1
    assert runs == 18

    # P = 8 (the smallest size the literal chain accepts): 16 spots per CTA, four per warp, reductions inside 8 lanes
    c8 = dataclasses.replace(W.CONFIGS[1], n=4, P=8, S=10, N=40, dx=0.2, screen_M=256)
    amp = W.pupil_mask(c8)
    yx = O.valid_list(amp, c8.n, c8.min_illum)
    ph = W.phase_frames(c8, 0, range(3))
    want, wimg = O.measure(ph, amp, yx, c8.n, c8.P, c8.b, tau=0.05, stage=2)
    for order in (0, 2):
        out = lit_run(exe, tmp_path, c8, 3, yx, 0, 0.05, ph, amp, None, 2, order, 8)
        assert out is not None
        compare(out[0], out[1], want, wimg, 0.05, 0, f"P = 8 order={order}")

    # without the barrier between the centred image written to shared memory and the binning that reads it
    mutant = harnesses["lit_mut"]
    c = small_config(3, 8)
    amp = W.pupil_mask(c)
    yx = O.valid_list(amp, c.n, c.min_illum)
    ph = W.phase_frames(c, 0, range(1))
    want, wimg = O.measure(ph, amp, yx, c.n, c.P, c.b, tau=0.1, stage=2)
    caught = 0
    for order in (0, 1, 2):
        out = lit_run(mutant, tmp_path, c, 1, yx, 0, 0.1, ph, amp, None, 2, order, 9)
        try:
            assert out is not None
            compare(out[0], out[1], want, wimg, 0.1, 0, "mutant")
        except AssertionError:
            caught += 1
    assert caught >= 1


# ---------------------------------------------------------------- pyramid.cu: the five kernels of a pyramid call

def pyr_extract(tmp_path: Path, mutate=None) -> None:
    src = (CSRC / "pyramid.cu").read_text()
    block = cut(src, "constexpr int PY_LINES = 8;", "template <int R>\ncudaError_t run_chunk")
    block, k1 = re.subn(r"extern __shared__ __align__\(16\) float2 py_smem\[\];",
                        "float2 *py_smem = reinterpret_cast<float2 *>(simt::smem());", block)
    block, k2 = re.subn(r"__shared__ float red\[256\];", "float *red = reinterpret_cast<float *>(simt::smem());", block)
    assert (k1, k2) == (3, 1) and "pyr_cols_kernel(const PyArgs A)" in block
    if mutate is not None:
        assert block.count(mutate[0]) == 1, mutate[0]
        block = block.replace(mutate[0], mutate[1])
    (tmp_path / "pyr_kernel_extract.inc").write_text(block)


def pyr_run(exe, tmp_path, ph, amp, yx, Np, s, bp, r_mod, K, D_pix, c_phi, order, seed):
    T, N, _ = ph.shape
    Sp = N // bp
    fin, fout = tmp_path / "in.bin", tmp_path / "out.bin"
    with open(fin, "wb") as f:
        f.write(struct.pack("10i", N, Np, s, bp, K, T, len(yx), order, seed, 0))
        f.write(struct.pack("3f", r_mod, D_pix, c_phi))
        f.write(np.ascontiguousarray(ph, np.float32).tobytes())
        f.write(np.ascontiguousarray(amp, np.float32).tobytes())
        f.write(np.ascontiguousarray(yx, np.int32).tobytes())
    r = subprocess.run([str(exe), str(fin), str(fout)], capture_output=True, text=True, timeout=900)
    if r.returncode != 0 or not r.stdout.startswith("ok "):
        assert r.stdout.startswith("FAIL"), r.stdout[-500:] + r.stderr[-500:]
        return None
    raw = np.fromfile(fout, np.float32)
    ns = T * len(yx) * 2
    return raw[:ns].reshape(T, len(yx), 2).astype(np.float64), raw[ns:].reshape(T, 2, 2, Sp, Sp).astype(np.float64)


def test_pyramid_kernels_whole_on_the_host(tmp_path, harnesses):
    from oracle import pyramid as OP
    exe = harnesses["pyr"]
    rng = np.random.default_rng(92)
    cases = []
    p = W.PYRAMIDS["tiny"]                                  # N = 48, Np = 256 (16 x 16 four-step), 8 modulation points
    cases.append((W.pyramid_frames(p, range(2)), W.pyramid_mask(p), p.Np, p.s, p.bp, p.r_mod, p.K, p.D_pix, 1.0, 0.5, (0, 1, 2)))
    # N not a multiple of the 8-line CTA, partially transmitting mask, phase_to_rad != 1, Np = 1024 (32 x 32 four-step)
    N = 44
    ax = np.arange(N) + 0.5 - N / 2
    amp = ((np.hypot(ax[None, :], ax[:, None]) <= N / 2) * rng.uniform(0.4, 1.0, (N, N))).astype(np.float32)
    cases.append((rng.normal(0, 2.0, (1, N, N)).astype(np.float32), amp, 1024, 200, 4, 1.5, 2, 0.9 * N, 0.6, 0.3, (2,)))
    # the LBT-like workload (240 x 240 pupil, Np = 1024, separation 256, 8 x 8 binning) with 4 of its 16
    # modulation points, one frame of its residual-like phase
    p = W.PYRAMIDS["lbt"]
    cases.append((W.pyramid_frames(p, range(1), 0.3), W.pyramid_mask(p), p.Np, p.s, p.bp, p.r_mod, 4, p.D_pix, 1.0, 0.5, (2,)))
    # unmodulated
    N = 36
    ax = np.arange(N) + 0.5 - N / 2
    amp = (np.hypot(ax[None, :], ax[:, None]) <= N / 2).astype(np.float32)
    cases.append((rng.normal(0, 1.0, (1, N, N)).astype(np.float32), amp, 256, 64, 2, 0.0, 0, float(N), 1.0, 0.5, (1,)))
    runs = 0
    for ph, amp, Np, s, bp, r_mod, K, D_pix, c_phi, min_illum, orders in cases:
        yx = OP.valid_pixels(amp, bp, min_illum)
        want, wq = OP.measure(ph, amp, yx, Np, s, bp, r_mod, K, D_pix, c_phi=np.float32(c_phi), return_quadrants=True)
        first = None
        for order in orders:
            label = f"pyramid N={ph.shape[-1]} Np={Np} K={K} order={order}"
            out = pyr_run(exe, tmp_path, ph, amp, yx, Np, s, bp, r_mod, K, D_pix, c_phi, order, 14 + runs)
            assert out is not None, label
            got, q = out
            assert not np.isnan(q).any() and not np.isnan(got).any(), label
            assert np.abs(q - wq).max() <= 1e-4 * wq.max(), (label, np.abs(q - wq).max() / wq.max())     # tests/test_pyramid_gpu.py
            assert np.abs(got - want).max() <= 2e-4, (label, np.abs(got - want).max())
            if first is None:
                first = out
            else:
                assert np.array_equal(first[0], got) and np.array_equal(first[1], q), f"{label}: depends on the thread order"
            runs += 1
    assert runs == 6

    # the exchange inside a line transform without its __syncwarp between the writes and the reads
    mutant = harnesses["pyr_mut"]
    ph, amp, Np, s, bp, r_mod, K, D_pix, c_phi, min_illum, _ = cases[3]
    yx = OP.valid_pixels(amp, bp, min_illum)
    want, wq = OP.measure(ph, amp, yx, Np, s, bp, r_mod, K, D_pix, c_phi=np.float32(c_phi), return_quadrants=True)
    caught = 0
    for order in (0, 1, 2):
        out = pyr_run(mutant, tmp_path, ph, amp, yx, Np, s, bp, r_mod, K, D_pix, c_phi, order, 3)
        if out is None or np.isnan(out[1]).any() or not np.abs(out[1] - wq).max() <= 1e-4 * wq.max():
            caught += 1
    assert caught >= 1


# ---------------------------------------------------------------- the paper's full LGS model on the EXT instances

def sodium_tables(c, yx, sod):
    """What shwfs_set_sodium (api.cu, host code, float64) puts into the handle: curvature per pixel^2, sqrt of the
    weights, and the local gradient of each sub-layer's analytic phase per subaperture, whole turns dropped."""
    two_pi = 2.0 * np.pi
    a = np.asarray(sod["defocus"], np.float64)
    yc = ((yx[:, 0] + 0.5) * c.n - 0.5 * c.N) * c.dx
    xc = ((yx[:, 1] + 0.5) * c.n - 0.5 * c.N) * c.dx
    gx = (2.0 * a[:, None] * (xc[None, :] - sod["cx"]) + np.asarray(sod["tilt_x"])[:, None]) * c.dx / two_pi
    gy = (2.0 * a[:, None] * (yc[None, :] - sod["cy"]) + np.asarray(sod["tilt_y"])[:, None]) * c.dx / two_pi
    g = np.stack([gx - np.rint(gx), gy - np.rint(gy)], axis=2).astype(np.float32)          # [L][nsub][2]
    return (a * c.dx * c.dx / two_pi).astype(np.float32), np.sqrt(np.asarray(sod["weight"])).astype(np.float32), g


def test_sodium_layers_and_noise_instances_whole_on_the_host(tmp_path, harnesses):
    """wk_measure_kernel<10,0,2> / <10,0,1> and wkf_kernel<10,0,2,ldg> / <10,0,1,ldg>: several sodium sub-layers with
    their own or a shared wavefront, and Gaussian-limit detector noise before the centroid (f2),
    against oracle/shwfs_oracle_lgs.c -- the MAORY geometry of config 3 at the real distance from the launch point."""
    exe = harnesses["wk"]
    c = small_config(3, 8)
    amp = W.pupil_mask(c)
    yx = O.valid_list(amp, c.n, c.min_illum)
    K = W.spot_size_kernels(c, yx)
    runs = 0
    for L, shared, T in ((3, False, 2), (5, True, 1)):
        sod = W.sodium_layers(W.CONFIGS[3], 0, L)              # launch point 19.5 m away: the elongation of the pupil edge
        ph = W.phase_frames(c, 0, range(T)) if shared else \
            np.stack([W.phase_frames(c, 0, range(10 * l, 10 * l + T)) for l in range(L)], axis=1)
        kw = dict(weight=sod["weight"], defocus=sod["defocus"], tilt_x=sod["tilt_x"], tilt_y=sod["tilt_y"],
                  cx=sod["cx"], cy=sod["cy"], tau=c.tau, kernels=K)
        want, wimg = O.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, stage=2, **kw)
        plain = O.measure(ph if shared else ph[:, 0], amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K)
        assert np.abs(want - plain).max() > 0.05                # the sub-layers do change the spots
        q, sw, g = sodium_tables(c, yx, sod)
        for kernel in ((0, 1, 2) if L == 3 else (0, 2)):      # 1: the size-generic kernel carries the sub-layers too
            first = None
            for order in ((2,) if kernel == 1 else (0, 2)):
                label = f"L={L} shared={shared} kernel={kernel} order={order}"
                out = wk_run(exe, tmp_path, c, T, yx, 0, c.tau, ph, amp, K, kernel, order, 31 + runs, L=L, sod_q=q, sod_sw=sw,
                             sod_g=g, shared=int(shared))
                assert out is not None, label
                compare(out[0], out[1], want, wimg, c.tau, 0, label)
                if first is None:
                    first = out
                else:
                    assert np.array_equal(first[0], out[0]) and np.array_equal(first[1], out[1]), label
                runs += 1
    # detector noise (Gaussian limit of the photon noise + read noise, Philox per (seed, t, i, pixel)) on 3 shared sub-layers
    L, T = 3, 2
    sod = W.sodium_layers(W.CONFIGS[3], 0, L)
    ph = W.phase_frames(c, 0, range(T))
    F, ron, seed = 500.0 / c.n ** 2, 3.0, 0x1408069800000091
    kw = dict(weight=sod["weight"], defocus=sod["defocus"], tilt_x=sod["tilt_x"], tilt_y=sod["tilt_y"],
              cx=sod["cx"], cy=sod["cy"], tau=c.tau, kernels=K)
    want, wimg = O.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, flux=F, ron=ron, seed=seed, stage=3, **kw)
    clean = O.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, **kw)
    assert np.abs(want - clean).max() > 0.05
    q, sw, g = sodium_tables(c, yx, sod)
    for kernel, Lk in ((0, L), (2, L), (0, 0)):
        if Lk == 0:                                             # noise on the plain single-layer sensor: instance <n,0,1>
            want, wimg = O.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, weight=[1.0], defocus=[0.0], tau=c.tau, kernels=K,
                                       flux=F, ron=ron, seed=seed, stage=3)
        out = wk_run(exe, tmp_path, c, T, yx, 0, c.tau, ph, amp, K, kernel, 2, 77, L=Lk, sod_q=q, sod_sw=sw,
                     sod_g=g if Lk else None, shared=1, flux=F, ron=ron, noise_seed=seed)
        assert out is not None
        label = f"noise kernel={kernel} L={Lk}"
        peak = wimg.max(axis=(2, 3), keepdims=True)
        assert float((np.abs(out[2] - wimg) / peak).max()) <= 1e-4, label
        assert float(np.abs(out[0] - want).max()) <= 1e-3, label
        runs += 1
    assert runs == 12


# ---------------------------------------------------------------- loop.cu: the closed-loop neighbours (FP32 kernels)

def loop_extract(tmp_path: Path, mutate=None) -> None:
    src = (CSRC / "loop.cu").read_text()
    block = src[src.index("/* modes[M][N][N] -> out[nsub][M][n*n]: block = (subaperture, mode) */"):
                src.index("}  // namespace\n\ncudaError_t shwfs_loop_relayout_modes")]
    block, k = re.subn(r"template <[^>]*>\nvoid launch_dm_\w+\(.*?\n}\n", "", block, flags=re.S)     # the launchers between the kernels
    assert k == 3 and "<<<" not in block
    block, k1 = re.subn(r"extern __shared__ __align__\(16\) float dm_smem\[\];", "float *dm_smem = reinterpret_cast<float *>(simt::smem());", block)
    block, k2 = re.subn(r"extern __shared__ float gv_coef\[\];", "float *gv_coef = reinterpret_cast<float *>(simt::smem());", block)
    block, k3 = re.subn(r"__shared__ float part\[RC_THREADS / 32\]\[RC_TT\];",
                        "float (*part)[RC_TT] = reinterpret_cast<float (*)[RC_TT]>(simt::smem());", block)
    assert (k1, k2, k3) == (1, 1, 1) and "recon_kernel(" in block and "dm_phase_kernel(" in block
    if mutate is not None:
        assert block.count(mutate[0]) == 1, mutate[0]
        block = block.replace(mutate[0], mutate[1])
    (tmp_path / "loop_kernel_extract.inc").write_text(block)


def loop_run(exe, tmp_path, c, yx, modes, coef, R, slopes, gain, variant, order, seed, lazy):
    T, M = coef.shape
    nsub = len(yx)
    fin, fout = tmp_path / "in.bin", tmp_path / "out.bin"
    with open(fin, "wb") as f:
        f.write(struct.pack("10i", c.N, c.n, nsub, M, T, variant, order, seed, lazy, M))
        f.write(struct.pack("f", gain))
        for a, dt in ((modes, np.float32), (yx, np.int32), (coef, np.float32), (R, np.float32), (slopes, np.float32)):
            f.write(np.ascontiguousarray(a, dt).tobytes())
    r = subprocess.run([str(exe), str(fin), str(fout)], capture_output=True, text=True, timeout=900)
    if r.returncode != 0 or not r.stdout.startswith("ok "):
        assert r.stdout.startswith("FAIL"), r.stdout[-500:] + r.stderr[-500:]
        return None
    raw = np.fromfile(fout, np.float32)
    npatch = T * nsub * c.n * c.n
    return (raw[:npatch].reshape(T, nsub, c.n, c.n).astype(np.float64), raw[npatch:npatch + T * M].reshape(T, M).astype(np.float64),
            raw[npatch + T * M:].reshape(T, M).astype(np.float64))


def test_closed_loop_kernels_whole_on_the_host(tmp_path, harnesses):
    """relayout_modes_kernel + dm_phase_kernel / dm_phase_gemv_kernel / dm_phase_simple_kernel against the definition
    C1 (oracle/closed_loop.py: the DM phase sum_m c[t,m] mode[m], here on the patches), recon_kernel against C2 and the
    integrator update, and the residual measured by wk_measure_kernel<10,0,1> / wkf_kernel<10,0,1,ldg> with that DM
    phase subtracted in the gather against oracle measure_residual."""
    from oracle import closed_loop as OL
    exe = harnesses["loop"]
    c = small_config(3, 8)
    amp = W.pupil_mask(c)
    yx = O.valid_list(amp, c.n, c.min_illum)
    nsub, M = len(yx), 37                                    # M neither a multiple of the 16-mode chunk nor of 8
    rng = np.random.default_rng(76)
    modes = W.dm_modes(c, M)
    R = rng.normal(0, 0.05, (M, 2 * nsub)).astype(np.float32)
    runs = 0
    for T, variant, lazy, orders in ((1, 0, 0, (2,)), (3, 0, 0, (1,)), (7, 1, 1, (0, 2)), (19, 0, 1, (0, 2)), (37, 1, 0, (2,)), (2, 2, 0, (2,))):
        coef = rng.normal(0, 0.5, (T, M)).astype(np.float32)
        slopes = rng.normal(0, 0.3, (T, 2 * nsub)).astype(np.float32)
        # C1 on the patches, float64
        full = np.einsum("tm,myx->tyx", coef.astype(np.float64), modes.astype(np.float64))
        want_patch = np.stack([full[:, sy * c.n:(sy + 1) * c.n, sx * c.n:(sx + 1) * c.n] for sy, sx in yx], axis=1)
        d = OL.reconstruct(R, slopes.reshape(T, nsub, 2))
        want_coef = coef.astype(np.float64) + 0.4 * d
        first = None
        for order in orders:
            label = f"T={T} variant={variant} lazy={lazy} order={order}"
            out = loop_run(exe, tmp_path, c, yx, modes, coef, R, slopes, 0.4, variant, order, 5 + runs, lazy)
            assert out is not None, label
            patch, coef_after, hist = out
            assert not np.isnan(patch).any(), label
            assert np.abs(patch - want_patch).max() <= 2e-5 * np.abs(want_patch).max(), (label, np.abs(patch - want_patch).max())
            assert np.array_equal(hist, coef.astype(np.float64)), label            # reading C4: the coefficients before the update
            assert np.abs(coef_after - want_coef).max() <= 1e-5, (label, np.abs(coef_after - want_coef).max())
            if first is None:
                first = out
            else:
                assert all(np.array_equal(a, b) for a, b in zip(first, out)), f"{label}: depends on the thread order"
            runs += 1
    assert runs == 8

    # the residual through the sensor: the DM phase of dm_phase_kernel subtracted in the gather (EXT instance)
    T = 2
    ph = W.phase_frames(c, 0, range(T))
    coef = rng.normal(0, 0.5, (T, M)).astype(np.float32)
    K = W.elongation_kernels(c, 0, yx)
    patch = loop_run(exe, tmp_path, c, yx, modes, coef, R, np.zeros((T, 2 * nsub), np.float32), 0.0, 1, 2, 3, 1)[0]
    want, wimg = OL.measure_residual(ph, modes, coef, amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K, stage=2)
    for kernel in (0, 2):
        out = wk_run(harnesses["wk"], tmp_path, c, T, yx, 0, c.tau, ph, amp, K, kernel, 2, 8, dm_patch=patch)
        assert out is not None
        compare(out[0], out[1], want, wimg, c.tau, 0, f"residual kernel={kernel}")

    # the double buffer of dm_phase_kernel without the barrier in front of its refill: with the copies completing as
    # late as the hardware may (lazy) and as early (eager), some thread order reads a stage another thread refills
    mutant = harnesses["loop_mut"]
    T = 19
    coef = rng.normal(0, 0.5, (T, M)).astype(np.float32)
    full = np.einsum("tm,myx->tyx", coef.astype(np.float64), modes.astype(np.float64))
    want_patch = np.stack([full[:, sy * c.n:(sy + 1) * c.n, sx * c.n:(sx + 1) * c.n] for sy, sx in yx], axis=1)
    caught = 0
    for order, lazy in ((0, 0), (1, 0), (2, 1)):
        out = loop_run(mutant, tmp_path, c, yx, modes, coef, R, np.zeros((T, 2 * nsub), np.float32), 0.0, 1, order, 3, lazy)
        if out is None or not np.abs(out[0] - want_patch).max() <= 2e-5 * np.abs(want_patch).max():
            caught += 1
    assert caught >= 1


@pytest.mark.parametrize("flux_total,ron", [(300.0, 0.0), (40000.0, 2.0)])
def test_poisson_noise_instance_whole_on_the_host(tmp_path, harnesses, flux_total, ron):
    """photon_model = 1 inside the kernels (add_noise_col16 of noise.cuh as wk_measure_kernel<10,0,1> and
    wkf_kernel<10,0,1,ldg> call it: pixel pairs, Philox counters and lanes as on the device), the statement of
    tests/test_lgs_gpu.py::test_config3_poisson_noise_matches_oracle: on every pixel whose draw the oracle reports as
    decided by more than rounding the count is the oracle's (exactly without read noise), the others differ by at most
    one count (inversion) or stay within 8 sigma (rejection), and spots whose image agrees have the oracle's slopes."""
    c = small_config(3, 8)
    amp = W.pupil_mask(c)
    yx = O.valid_list(amp, c.n, c.min_illum)
    K = W.elongation_kernels(c, 0, yx)
    T = 2
    ph = W.phase_frames(c, 0, range(T))
    F, seed = flux_total / c.n ** 2, 0x14080698000000A7
    kw = dict(weight=[1.0], defocus=[0.0], tau=c.tau, kernels=K, flux=F, ron=ron, seed=seed, photon_model=1)
    want, wimg, margin = O.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, stage=3, want_margins=True, **kw)
    _, clean_img = O.measure_lgs(ph, amp, yx, c.n, c.P, c.b, c.dx, weight=[1.0], defocus=[0.0], tau=c.tau, kernels=K, stage=2)
    rate = np.maximum(F * clean_img, 0.0)
    assert (rate >= 30).any() == (flux_total > 1000)                  # which branch the case exercises
    clear = margin > 1e-4 + 1e-5 * rate                               # _poisson_clear of tests/test_lgs_gpu.py
    assert clear.mean() > 0.95
    for kernel in (0, 2):
        out = wk_run(harnesses["wk"], tmp_path, c, T, yx, 0, c.tau, ph, amp, K, kernel, 2, 21, flux=F, ron=ron,
                     noise_seed=seed, photon_model=1)
        assert out is not None
        got, _, img = out
        d = np.abs(img - wimg)
        if ron == 0.0:
            assert np.all(img == np.round(img)) and img.min() >= 0
            assert np.all(d[clear] == 0.0), (kernel, d[clear].max(), int((d[clear] > 0).sum()))
        else:
            pk = wimg.max(axis=(2, 3), keepdims=True)
            assert (d / pk)[clear].max() <= 1e-4, (kernel, (d / pk)[clear].max())
        low = ~clear & (rate < 29.9)
        assert d[low].max(initial=0.0) <= 1.0 + 1e-3
        high = ~clear & (rate >= 29.9)
        assert np.all(d[high] <= 8.0 * np.sqrt(rate[high]) + 2.0)
        same = (d <= (1e-6 if ron == 0.0 else 1e-4 * wimg.max(axis=(2, 3), keepdims=True))).all(axis=(2, 3))
        assert same.mean() > 0.05
        assert np.abs(got - want)[same].max() <= 1e-3, (kernel, np.abs(got - want)[same].max())
        assert (d > 0.5).mean() <= 2.0 * (~clear).mean() + 1e-4


def test_config3_whole_frame_headline_kernel_on_the_host(tmp_path, harnesses):
    """One whole frame of config 3 (BASELINE.json:configs[2], one WFS of the headline config 4): the real 800 x 800 pupil,
    its 4632 valid subapertures with their radially elongated kernels, in the launch shape the library uses (145 CTAs of
    32 spots, the last one ragged), through wk_table_kernel + wk_measure_kernel<10,0,0>: EVERY spot against the oracle."""
    c = W.CONFIGS[3]
    amp = W.pupil_mask(c)
    yx = O.valid_list(amp, c.n, c.min_illum)
    assert len(yx) == 4632
    ph = W.phase_frames(c, 0, range(1))
    K = W.elongation_kernels(c, 0, yx)
    want, wimg = O.measure(ph, amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K, stage=2)
    out = wk_run(harnesses["wk"], tmp_path, c, 1, yx, 0, c.tau, ph, amp, K, 0, 2, 4)
    assert out is not None
    ierr, serr = compare(out[0], out[1], want, wimg, c.tau, 0, "config 3, whole frame")
    assert ierr <= 2e-6 and serr <= 2e-5            # measured 3.4e-7 of the peak and 1.3e-6 px: two orders inside the tolerances


def test_config2_whole_frame_pruned_fft_kernel_on_the_host(tmp_path, harnesses):
    """One whole frame of config 2 (BASELINE.json:configs[1]): the real 640 x 640 pupil with its 20 % obstruction, every
    valid subaperture, through pruned_fft_kernel<32,16,0,tma> as a persistent launch of 8 CTAs with the dynamic deal
    (chunks of four spots from the counter, boxes completed as late as the hardware may): EVERY spot against the oracle."""
    c = W.CONFIGS[2]
    amp = W.pupil_mask(c)
    yx = O.valid_list(amp, c.n, c.min_illum)
    ph = W.phase_frames(c, 0, range(1))
    table = patch_table(amp, yx, c.n)
    lit = (table[:, 0] & PATCH_LIT) != 0
    assert 0.85 < lit.mean() < 0.98                                   # "93 % of config 2" read no amplitude (pruned_fft.cu)
    want, wimg = O.measure(ph, amp, yx, c.n, c.P, c.b, tau=c.tau, stage=2)
    out = pf_run(harnesses["pf"], tmp_path, c, 1, len(yx), 0, c.tau, ph, amp, table, 1, 4, 1, 8, 2, 11)
    assert out is not None
    words = out[2].split()
    assert int(words[words.index("boxes") + 1]) == len(yx)
    ierr, serr = compare(out[0], out[1], want, wimg, c.tau, 0, "config 2, whole frame")
    assert ierr <= 5e-6 and serr <= 5e-5


def test_config5_frame_subset_fft_kernel_on_the_host(tmp_path, harnesses):
    """Config 5 (BASELINE.json:configs[4]: 1280 x 1280 pupil, n = 16, P = 64, 4 x 4 binning, kernels up to 6 arcsec) at its
    real geometry, every seventh valid subaperture of one frame (pupil edge, obstruction edge and interior alike) with its
    own elongation kernel, through wkf_kernel<16,0,0,tma> as a persistent launch of 3 CTAs with the dynamic deal."""
    c = W.CONFIGS[5]
    amp = W.pupil_mask(c)
    yx = O.valid_list(amp, c.n, c.min_illum)[::7].copy()
    ph = W.phase_frames(c, 0, range(1))
    K = W.elongation_kernels(c, 0, yx)
    want, wimg = O.measure(ph, amp, yx, c.n, c.P, c.b, tau=c.tau, kernels=K, stage=2)
    out = wk_run(harnesses["wk"], tmp_path, c, 1, yx, 0, c.tau, ph, amp, K, 3, 2, 12, grid=3, lazy=1)
    assert out is not None
    ierr, serr = compare(out[0], out[1], want, wimg, c.tau, 0, "config 5, one frame, every 7th subaperture")
    assert ierr <= 5e-6 and serr <= 5e-5


def test_tensor_core_operand_preparation_on_the_host(tmp_path):
    """dm_umma.cu's operand kernels (TF32 hi/lo split into canonical K-major tiles) on the host SIMT machine
    (tests/host/umma_prep_harness.cpp): layout, padding, TF32-ness, and the 3-term product summed exactly from the
    tiles against the plain GEMM -- DESIGN.md 6.5's figures for the split (1.7e-7 of peak) and a single pass (4.9e-4)."""
    if shutil.which("g++") is None or not (CUDA_INC / "cuda_runtime.h").exists():
        pytest.skip("needs g++ and the CUDA headers")
    src = (CSRC / "dm_umma.cu").read_text()
    block = cut(src, "constexpr int UM_KB = 8;", "__device__ __forceinline__ uint64_t umma_desc(")
    block, k = re.subn(r"    uint32_t r;\n    asm\(\"cvt\.rna\.tf32\.f32 %0, %1;\" : \"=r\"\(r\) : \"f\"\(x\)\);\n    return __uint_as_float\(r\);\n",
                       "    return host_tf32_rna(x);\n", block)
    assert k == 1 and "umma_split_modes_kernel(" in block and "umma_split_coef_kernel(" in block and "asm" not in block
    (tmp_path / "umma_prep_extract.inc").write_text(block)
    exe = tmp_path / "umma_prep_harness"
    r = subprocess.run(["g++", "-std=c++17", "-O1", "-ffp-contract=off", f"-I{CUDA_INC}", f"-I{tmp_path}", "-Wno-attributes", "-Wno-psabi",
                        "-o", str(exe), str(ROOT / "tests" / "host" / "umma_prep_harness.cpp")], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    # (nsub, M, n*n, padded n*n, frames): the three sizes with an instance; M and T ragged against the 8-mode stage / 128-frame tile
    for args in ((5, 37, 100, 112, 150), (3, 16, 64, 64, 128), (2, 21, 256, 256, 9)):
        run = subprocess.run([str(exe), *map(str, args)], capture_output=True, text=True, timeout=600)
        assert run.returncode == 0 and run.stdout.startswith("ok "), (args, run.stdout[-500:] + run.stderr[-500:])
        split, single = (float(w) for w in run.stdout.split()[1:3])
        assert split <= 5e-7, (args, split)                  # fp32-class: the dropped lo x lo term and the lo roundings
        assert 5e-5 <= single <= 2e-3, (args, single)        # what one TF32 pass would have given

"""The C ABI: exported symbols and struct layout (CPU), argument checking and handle life cycle (GPU)."""
import ctypes as C
import re
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent
HEADER = ROOT / "include" / "shwfs.h"


def _declared_functions():
    text = re.sub(r"/\*.*?\*/", "", HEADER.read_text(), flags=re.S)
    return sorted(set(re.findall(r"\b(shwfs_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(libshwfs):
    from paper_1408_0698_b200 import binding
    names = _declared_functions()
    assert "shwfs_create" in names and "shwfs_measure" in names and "shwfs_destroy" in names
    lib = C.CDLL(str(libshwfs))
    for name in names:
        assert hasattr(lib, name), f"{name} is declared in include/shwfs.h but not exported"
    assert sorted(binding.EXPORTS) == names
    L = binding.load()
    assert L.shwfs_version() >= 100
    assert L.shwfs_strerror(0) == b"ok"
    assert b"invalid" in L.shwfs_strerror(-1)


def test_binding_constants_match_the_header():
    """Every #define of include/shwfs.h with an integer value (error codes, SHWFS_ALGO_*, SHWFS_MAX_LAYERS) has
    the same value in the binding (ALGO_* drop the SHWFS_ prefix there)."""
    from paper_1408_0698_b200 import binding
    defs = dict(re.findall(r"^#define\s+(SHWFS_[A-Z_]+)\s+\(?(-?\d+)\)?", HEADER.read_text(), flags=re.M))
    assert {"SHWFS_OK", "SHWFS_ECUDA", "SHWFS_ALGO_AUTO", "SHWFS_ALGO_WK_FFT", "SHWFS_MAX_LAYERS"} <= set(defs)
    for name, value in defs.items():
        py = name[len("SHWFS_"):] if name.startswith("SHWFS_ALGO_") else name
        assert getattr(binding, py) == int(value), name
    algos = sorted(int(v) for k, v in defs.items() if k.startswith("SHWFS_ALGO_"))
    assert algos == list(range(len(algos)))                 # dense, no two algorithms share a number


@pytest.mark.parametrize("cname,pyname", [("shwfs_geometry", "ShwfsGeometry"), ("shwfs_sodium", "ShwfsSodium"),
                                          ("shwfs_noise", "ShwfsNoise"), ("pyrwfs_config", "PyrwfsConfig")])
def test_ctypes_struct_matches_the_header(tmp_path, cname, pyname):
    """sizeof / offsetof of each ABI struct as gcc sees the header == the ctypes mirror in the binding."""
    from paper_1408_0698_b200 import binding
    St = getattr(binding, pyname)
    fields = [f[0] for f in St._fields_]
    src = tmp_path / "layout.c"
    body = "".join(f'printf("%zu\\n", offsetof({cname}, {f}));' for f in fields)
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "shwfs.h"\n#include "pyrwfs.h"\n'
                   f'int main(void){{printf("%zu\\n", sizeof({cname}));' + body + "return 0;}\n")
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-std=c99", "-I", str(ROOT / "include"), str(src), "-o", str(exe)], check=True)
    out = [int(v) for v in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()]
    assert out[0] == C.sizeof(St)
    assert out[1:] == [getattr(St, f).offset for f in fields]


def test_library_exports_every_pyramid_symbol(libshwfs):
    from paper_1408_0698_b200 import binding
    text = re.sub(r"/\*.*?\*/", "", (ROOT / "include" / "pyrwfs.h").read_text(), flags=re.S)
    names = sorted(set(re.findall(r"\b(pyrwfs_[a-z_]+)\s*\(", text)))
    lib = C.CDLL(str(libshwfs))
    for name in names:
        assert hasattr(lib, name), f"{name} is declared in include/pyrwfs.h but not exported"
    assert sorted(binding.PYR_EXPORTS) == names


def test_header_compiles_as_c_and_cxx(tmp_path):
    for comp, ext in (("gcc", "c"), ("g++", "cpp")):
        src = tmp_path / f"inc.{ext}"
        src.write_text('#include "shwfs.h"\nint main(void){return SHWFS_OK;}\n')
        subprocess.run([comp, "-Wall", "-Werror", "-I", str(ROOT / "include"), "-c", str(src), "-o",
                        str(tmp_path / f"inc_{ext}.o")], check=True)


def test_no_cpu_fallback(libshwfs):
    """Without a CUDA device the product path raises; it never routes anywhere else."""
    import torch
    from paper_1408_0698_b200 import binding, workloads as W
    if torch.cuda.is_available():
        pytest.skip("this box has a GPU")
    c = W.CONFIGS[1]
    with pytest.raises(RuntimeError, match="CUDA device"):
        binding.from_config(c, 0)
    # and the raw C call reports a CUDA error instead of computing anything
    g = binding.ShwfsGeometry()
    amp = W.pupil_mask(c)
    g.n_pupil, g.n_sub_side, g.n_pix, g.pixel_size_m = c.N, c.S, c.n, c.dx
    g.amplitude = amp.ctypes.data_as(C.POINTER(C.c_float))
    g.min_illum, g.threshold_frac, g.threshold_mode, g.phase_to_rad = 0.5, 0.0, 0, 1.0
    with pytest.raises(binding.ShwfsError) as ei:
        binding.shwfs_create(g, W.LAMBDA_M, c.P, c.b)
    assert ei.value.code in (binding.SHWFS_ECUDA, binding.SHWFS_ENOMEM)


def test_product_does_not_import_the_oracle():
    """oracle/ is test infrastructure: nothing under the package may import, load or name it."""
    pkg = ROOT / "paper_1408_0698_b200"
    for p in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")) + list(pkg.rglob("*.h")):
        text = p.read_text()
        assert "shwfs_oracle" not in text and "from oracle" not in text and "import oracle" not in text, p
    for p in (ROOT / "oracle").glob("*"):
        if p.suffix in (".py", ".c", ".h"):
            assert "paper_1408_0698_b200" not in p.read_text().replace("imports nothing from paper_1408_0698_b200", "") \
                .replace("under paper_1408_0698_b200/csrc/", ""), p


# ------------------------------------------------------------------------------------------- GPU

def _geom(binding, c, amp, **kw):
    g = binding.ShwfsGeometry()
    g.n_pupil, g.n_sub_side, g.n_pix, g.pixel_size_m = c.N, c.S, c.n, c.dx
    g.amplitude = amp.ctypes.data_as(C.POINTER(C.c_float))
    g.min_illum, g.threshold_frac, g.threshold_mode, g.phase_to_rad = 0.5, 0.0, 0, 1.0
    for k, v in kw.items():
        setattr(g, k, v)
    return g


@pytest.mark.gpu
def test_create_rejects_bad_arguments(gpu):
    torch, B = gpu
    from paper_1408_0698_b200 import workloads as W
    c = W.CONFIGS[1]
    amp = W.pupil_mask(c)
    L = B.load()
    out = C.c_void_p(0xDEAD)

    def rc(g, lam=W.LAMBDA_M, P=c.P, b=c.b, k=None, o=out):
        return L.shwfs_create(C.byref(g) if g is not None else None, lam, P, b, k, C.byref(o) if o is not None else None)

    assert rc(None) == B.SHWFS_EINVAL
    assert rc(_geom(B, c, amp), o=None) == B.SHWFS_EINVAL
    assert rc(_geom(B, c, amp, n_sub_side=9)) == B.SHWFS_EINVAL          # N != S*n
    assert rc(_geom(B, c, amp), P=24) == B.SHWFS_EINVAL                  # not a power of two
    assert rc(_geom(B, c, amp), P=4) == B.SHWFS_EINVAL                   # n > P
    assert rc(_geom(B, c, amp), P=128) == B.SHWFS_EINVAL
    assert rc(_geom(B, c, amp), b=3) == B.SHWFS_EINVAL                   # b does not divide P
    assert rc(_geom(B, c, amp), b=16) == B.SHWFS_EINVAL                  # (P/2) % b != 0
    assert rc(_geom(B, c, amp), lam=0.0) == B.SHWFS_EINVAL
    assert rc(_geom(B, c, amp, pixel_size_m=0.0)) == B.SHWFS_EINVAL
    assert rc(_geom(B, c, amp, threshold_frac=1.0)) == B.SHWFS_EINVAL
    assert rc(_geom(B, c, amp, threshold_mode=2)) == B.SHWFS_EINVAL
    assert rc(_geom(B, c, amp, min_illum=2.0)) == B.SHWFS_EINVAL         # no valid subaperture
    bad = np.array([[0, 10]], dtype=np.int32)
    assert rc(_geom(B, c, amp, valid_yx=bad.ctypes.data_as(C.POINTER(C.c_int32)), n_valid=1)) == B.SHWFS_EINVAL
    g = _geom(B, c, amp)
    g.amplitude = None
    assert rc(g) == B.SHWFS_EINVAL
    assert out.value == 0xDEAD                                           # untouched on failure
    assert L.shwfs_destroy(None) == B.SHWFS_OK


@pytest.mark.gpu
def test_measure_rejects_bad_arguments_and_queries(gpu):
    torch, B = gpu
    from paper_1408_0698_b200 import workloads as W
    c = W.CONFIGS[1]
    L = B.load()
    with B.from_config(c, 0) as s:
        ph = torch.zeros((2, c.N, c.N), dtype=torch.float32, device="cuda")
        out = torch.zeros((2, s.nsub, 2), dtype=torch.float32, device="cuda")
        assert L.shwfs_measure(None, ph.data_ptr(), 2, out.data_ptr(), None) == B.SHWFS_EINVAL
        assert L.shwfs_measure(s._h, None, 2, out.data_ptr(), None) == B.SHWFS_EINVAL
        assert L.shwfs_measure(s._h, ph.data_ptr(), 2, None, None) == B.SHWFS_EINVAL
        assert L.shwfs_measure(s._h, ph.data_ptr(), -1, out.data_ptr(), None) == B.SHWFS_EINVAL
        assert L.shwfs_measure(s._h, None, 0, None, None) == B.SHWFS_OK
        assert L.shwfs_debug_spots(s._h, ph.data_ptr(), 2, 4, out.data_ptr(), None) == B.SHWFS_EINVAL
        assert L.shwfs_set_algorithm(s._h, 99) == B.SHWFS_EINVAL
        assert L.shwfs_num_subaps(s._h, None) == B.SHWFS_EINVAL
        assert s.nsub == 80
        assert abs(s.pixel_scale - c.b * W.LAMBDA_M / (c.P * c.dx)) < 1e-12   # float dx, lambda
        assert s.algorithm in (B.ALGO_LITERAL, B.ALGO_WK, B.ALGO_WK_GENERIC, B.ALGO_PRUNED_FFT, B.ALGO_WK_FFT)
        yx = s.valid_yx
        assert yx.shape == (80, 2) and (np.diff(yx[:, 0] * c.S + yx[:, 1]) > 0).all()   # row-major order


@pytest.mark.gpu
def test_two_handles_two_streams_and_repeatability(gpu, oracle):
    torch, B = gpu
    from paper_1408_0698_b200 import workloads as W
    c = W.CONFIGS[3]
    dev = torch.device("cuda")
    a, b = B.from_config(c, 0), B.from_config(c, 2)
    try:
        pa, pb = (W.phase_frames_device(c, w, range(8), dev) for w in (0, 2))
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        torch.cuda.synchronize()
        r1 = [a.measure(pa, stream=s1) for _ in range(3)]
        r2 = [b.measure(pb, stream=s2) for _ in range(3)]
        torch.cuda.synchronize()
        for r in r1[1:]:
            assert torch.equal(r, r1[0])                 # deterministic: no atomics, fixed reduction order
        for r in r2[1:]:
            assert torch.equal(r, r2[0])
        assert not torch.equal(r1[0], r2[0])
        # create / destroy loop leaves no residue that changes results
        for _ in range(3):
            with B.from_config(c, 0) as t:
                assert torch.equal(t.measure(pa), r1[0])
    finally:
        a.close(); b.close()


@pytest.mark.gpu
@pytest.mark.parametrize("pinned", [False, True])
def test_measure_host_matches_device_path(gpu, pinned):
    """Host-buffer entry point: several chunks (T larger than one 64 MiB chunk), pageable and pinned."""
    torch, B = gpu
    from paper_1408_0698_b200 import workloads as W
    c = W.CONFIGS[2]                                     # 1.6 MB frames -> 40-frame chunks
    with B.from_config(c, 0) as s:
        T = 97
        dev = torch.device("cuda")
        phd = W.phase_frames_device(c, 0, range(T), dev)
        want = s.measure(phd).cpu()
        host = torch.empty((T, c.N, c.N), dtype=torch.float32, pin_memory=pinned)
        host.copy_(phd)
        got = s.measure_host(host)
        assert torch.equal(got, want)
        got_np = s.measure_host(host.numpy())
        np.testing.assert_array_equal(got_np, want.numpy())
        got2 = s.measure_host(host[:3].contiguous())      # smaller call after a larger one
        assert torch.equal(got2, want[:3])


def test_library_carries_blackwell_tensor_core_code(libshwfs):
    """The DM-phase GEMM is tcgen05 code: the SASS of the built library holds UTCHMMA (tcgen05.mma), LDTM
    (tcgen05.ld) and UBLKCP (cp.async.bulk) -- the mnemonics of B200_PROFILING.md -- and no legacy HMMA path."""
    import shutil
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not Path(cuobjdump).exists():
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([cuobjdump, "-sass", str(libshwfs)], capture_output=True, text=True, check=True).stdout
    assert "UTCHMMA" in sass and "LDTM" in sass and "UBLKCP" in sass
    assert "HGMMA" not in sass and " HMMA" not in sass
    assert "sm_100a" in sass


@pytest.mark.gpu
def test_measure_host_async_matches_the_blocking_call(gpu):
    torch, B = gpu
    from paper_1408_0698_b200 import workloads as W
    c = W.CONFIGS[1]
    host = torch.from_numpy(W.phase_frames(c, 0, range(4))).pin_memory()
    with B.from_config(c, 0) as s1, B.from_config(c, 0) as s2:
        want = s1.measure_host(host).clone()
        o1 = torch.empty((4, s1.nsub, 2), dtype=torch.float32).pin_memory()
        o2 = torch.empty((4, s2.nsub, 2), dtype=torch.float32).pin_memory()
        s1.measure_host_async(host, o1)
        s2.measure_host_async(host, o2)               # two handles in flight
        s1.host_wait(); s2.host_wait()
        assert torch.equal(o1, want) and torch.equal(o2, want)
        rc = B.load().shwfs_measure_host_async(s1._h, host.numpy().copy().ctypes.data, 4, o1.data_ptr())
        assert rc == B.SHWFS_EINVAL                   # pageable input is refused

"""The device code around the autocorrelation in the lag-domain path -- wk_table_kernel of csrc/wk.cu (H0, the table M,
cut out of the .cu file as text and run with one simulated thread per block), csrc/field.cuh (H2), csrc/wk_common.cuh
(table product, x- and y-transform: H5 + H6 in Fourier form), csrc/cog.cuh (H7 + H8, shuffles simulated) -- compiled
as it is for the host and compared with the float64 oracle's chain O2..O9 (tests/host/lagdomain_harness.cpp) at the
sizes of configs 1, 2, 3/4 and 5, with and without elongation kernels, both threshold modes, phases up to +-60 rad:
binned images within 1e-4 of the peak, slopes within 1e-3 px (north_star).  CPU-side parity of device code: no GPU."""
import shutil
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
CUDA_INC = Path("/usr/local/cuda/include")


@pytest.mark.skipif(shutil.which("g++") is None or shutil.which("gcc") is None
                    or not (CUDA_INC / "cuda_runtime.h").exists(), reason="needs gcc, g++ and the CUDA headers")
def test_lag_domain_device_code_matches_the_oracle_on_the_host(tmp_path):
    # H0: the table kernel of wk.cu, cut out as text (the kernels after it use launch syntax g++ cannot read)
    src = (ROOT / "paper_1408_0698_b200" / "csrc" / "wk.cu").read_text()
    begin, end = "__global__ void wk_table_kernel(", "/* ------------------------------------------------------------------------------------------------\n * Specialised kernel:"
    assert src.count(begin) == 1 and src.count(end) == 1, "markers of wk_table_kernel not found in wk.cu"
    block = src[src.index(begin):src.index(end)]
    assert "<<<" not in block and block.count("__global__") == 1 and "sincospi" in block
    (tmp_path / "wk_table_extract.inc").write_text(block)
    obj = tmp_path / "shwfs_oracle.o"
    r = subprocess.run(["gcc", "-O2", "-std=c99", "-fopenmp", "-ffp-contract=off", "-c",
                        str(ROOT / "oracle" / "shwfs_oracle.c"), "-o", str(obj)], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr[-2000:]
    exe = tmp_path / "lagdomain_harness"
    build = subprocess.run(["g++", "-std=c++17", "-O1", "-ffp-contract=off", f"-I{CUDA_INC}", f"-I{tmp_path}", "-Wno-attributes",
                            "-o", str(exe), str(ROOT / "tests" / "host" / "lagdomain_harness.cpp"), str(obj), "-lm",
                            "-fopenmp"], capture_output=True, text=True, timeout=600)
    assert build.returncode == 0, build.stderr[-2000:]
    run = subprocess.run([str(exe)], capture_output=True, text=True, timeout=600)
    assert run.returncode == 0 and run.stdout.startswith("ok "), run.stdout[-2000:] + run.stderr[-2000:]
    words = run.stdout.split()
    assert float(words[words.index("error") + 1]) <= 1e-4           # images, of the peak
    assert float(words[-2]) <= 1e-3                                  # slopes, px

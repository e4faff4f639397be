"""The four-step line transform of the pyramid sensor (csrc/pyramid.cu: unscramble, cmul2, PowWalk, line_fft) cut out of
the .cu file as it is, compiled for the host (the R threads of a line run in two passes in place of the __syncwarp)
and compared with a float64 DFT of length 256 and 1024, both signs, full and input-pruned
(tests/host/pyr_line_harness.cpp).  Host logic: no GPU."""
import shutil
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
CUDA_INC = Path("/usr/local/cuda/include")
BEGIN = "/* natural-order copy of a transform result: out[k] = X[k] */"
END = "/* index of pupil-plane coordinate c (row or column) among the 2N kept ones"


@pytest.mark.skipif(shutil.which("g++") is None or not (CUDA_INC / "cuda_runtime.h").exists(),
                    reason="needs g++ and the CUDA headers")
def test_four_step_line_transform_matches_a_float64_dft(tmp_path):
    src = (ROOT / "paper_1408_0698_b200" / "csrc" / "pyramid.cu").read_text()
    assert src.count(BEGIN) == 1 and src.count(END) == 1, "markers of the line-transform block not found in pyramid.cu"
    block = src[src.index(BEGIN):src.index(END)]
    for name in ("struct PowWalk", "void line_fft(", "float2 cmul2(", "void unscramble("):
        assert name in block, name
    assert "<<<" not in block and "__global__" not in block
    (tmp_path / "pyr_line_extract.inc").write_text(block)
    exe = tmp_path / "pyr_line_harness"
    build = subprocess.run(["g++", "-std=c++17", "-O0", "-ffp-contract=off", f"-I{CUDA_INC}", f"-I{tmp_path}",
                            "-Wno-attributes", "-o", str(exe), str(ROOT / "tests" / "host" / "pyr_line_harness.cpp")],
                           capture_output=True, text=True, timeout=900)
    assert build.returncode == 0, build.stderr[-2000:]
    run = subprocess.run([str(exe)], capture_output=True, text=True, timeout=300)
    assert run.returncode == 0 and run.stdout.startswith("ok "), run.stdout[-2000:] + run.stderr[-2000:]

"""csrc/fft_regs.cuh -- the register-resident line transforms every kernel uses -- compiled as it is for the host
(tests/host/fft_regs_harness.cpp; the FP32x2 intrinsics shimmed component-wise) and checked against a float64 DFT
for L = 2..64, both signs, full and pruned inputs; the packed transform must equal the scalar one bit for bit, as
the header says, and the split-first-stage form the packed one.  Host logic: no GPU."""
import shutil
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
CUDA_INC = Path("/usr/local/cuda/include")


@pytest.mark.skipif(shutil.which("g++") is None or not (CUDA_INC / "cuda_runtime.h").exists(),
                    reason="needs g++ and the CUDA headers")
def test_register_ffts_match_a_float64_dft(tmp_path):
    exe = tmp_path / "fft_regs_harness"
    build = subprocess.run(["g++", "-std=c++17", "-O0", "-ffp-contract=off", f"-I{CUDA_INC}", "-Wno-attributes",
                            "-o", str(exe), str(ROOT / "tests" / "host" / "fft_regs_harness.cpp")],
                           capture_output=True, text=True, timeout=600)
    assert build.returncode == 0, build.stderr[-2000:]
    run = subprocess.run([str(exe)], capture_output=True, text=True, timeout=300)
    assert run.returncode == 0 and run.stdout.startswith("ok "), run.stdout[-2000:] + run.stderr[-2000:]
    worst = float(run.stdout.split("worst error")[1].split()[0])
    assert worst <= 5e-7          # <= 4.5e-7 on unit-range data

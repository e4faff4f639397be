"""csrc/sweep.cuh -- the deal of spots to the warps of the persistent kernels -- compiled as it is for the host and
run over 1200 simulated launches (tests/host/sweep_harness.cpp): every spot visited exactly once with the right
(subaperture, frame) and table entry, under the strided and the dynamic deal, on ragged shapes, with warps running at
unequal speeds, two launches in a row on one counter.  Host logic: no GPU."""
import shutil
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
CUDA_INC = Path("/usr/local/cuda/include")


@pytest.mark.skipif(shutil.which("g++") is None or not (CUDA_INC / "cuda_runtime.h").exists(),
                    reason="needs g++ and the CUDA headers")
def test_every_spot_is_dealt_exactly_once(tmp_path):
    exe = tmp_path / "sweep_harness"
    build = subprocess.run(["g++", "-std=c++17", "-O1", f"-I{CUDA_INC}", "-Wno-attributes", "-o", str(exe),
                            str(ROOT / "tests" / "host" / "sweep_harness.cpp")], capture_output=True, text=True)
    assert build.returncode == 0, build.stderr[-2000:]
    run = subprocess.run([str(exe)], capture_output=True, text=True, timeout=300)
    assert run.returncode == 0 and run.stdout.startswith("ok "), run.stdout[-2000:] + run.stderr[-2000:]
    launches = int(run.stdout.split()[1])
    assert launches > 1000

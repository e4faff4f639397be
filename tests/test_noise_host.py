"""csrc/noise.cuh -- detector noise before the centroid -- compiled as it is for the host and
compared with the float64 oracle's C functions (tests/host/noise_harness.cpp): Philox4x32-10 bit for bit, the normal
deviates, the Gaussian-limit counts, and the fp32 Poisson draw (inversion / PTRS), whose integer must be the oracle's
on every draw the oracle reports as decided by more than rounding -- the criterion of tests/test_lgs_gpu.py, here on
100 000 draws over rates from 0.02 to 2500.  CPU-side parity of device code: no GPU."""
import shutil
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
CUDA_INC = Path("/usr/local/cuda/include")


@pytest.mark.skipif(shutil.which("g++") is None or shutil.which("gcc") is None
                    or not (CUDA_INC / "cuda_runtime.h").exists(), reason="needs gcc, g++ and the CUDA headers")
def test_device_noise_code_matches_the_oracle_on_the_host(tmp_path):
    objs = []
    for src in ("shwfs_oracle.c", "shwfs_oracle_lgs.c", "shwfs_oracle_poisson.c"):      # the oracle as it stands
        obj = tmp_path / (src + ".o")
        r = subprocess.run(["gcc", "-O2", "-std=c99", "-fopenmp", "-ffp-contract=off", "-c", str(ROOT / "oracle" / src),
                            "-o", str(obj)], capture_output=True, text=True)
        assert r.returncode == 0, r.stderr[-2000:]
        objs.append(str(obj))
    exe = tmp_path / "noise_harness"
    build = subprocess.run(["g++", "-std=c++17", "-O1", "-ffp-contract=off", f"-I{CUDA_INC}", "-Wno-attributes",
                            "-o", str(exe), str(ROOT / "tests" / "host" / "noise_harness.cpp"), *objs, "-lm", "-fopenmp"],
                           capture_output=True, text=True, timeout=600)
    assert build.returncode == 0, build.stderr[-2000:]
    run = subprocess.run([str(exe)], capture_output=True, text=True, timeout=300)
    assert run.returncode == 0 and run.stdout.startswith("ok "), run.stdout[-2000:] + run.stderr[-2000:]
    clear = int(run.stdout.split(",")[2].split()[0])
    assert clear > 90000

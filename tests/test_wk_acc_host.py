"""The autocorrelation accumulators of the headline kernel (csrc/wk.cu: LagAcc, rowpair_acc, rowself_acc -- the
three-real-product complex MAC on packed FFMA2) cut out of the .cu file as they are, compiled for the host and compared
with the plain double sums of G[ly,lx] = sum e[j,k] conj(e[j+ly,k+lx]) (tests/host/wk_acc_harness.cpp) for n = 8, 10,
16.  Host logic: no GPU."""
import shutil
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
CUDA_INC = Path("/usr/local/cuda/include")
BEGIN = "template <int n>\n__device__ __forceinline__ void load_row("
END = "/* EXTK: 0 = plain sensor;"


@pytest.mark.skipif(shutil.which("g++") is None or not (CUDA_INC / "cuda_runtime.h").exists(),
                    reason="needs g++ and the CUDA headers")
def test_three_product_autocorrelation_matches_plain_sums(tmp_path):
    src = (ROOT / "paper_1408_0698_b200" / "csrc" / "wk.cu").read_text()
    assert src.count(BEGIN) == 1 and src.count(END) == 1, "markers of the accumulator block not found in wk.cu"
    block = src[src.index(BEGIN):src.index(END)]
    for name in ("struct LagAcc", "void rowpair_acc(", "void rowself_acc(", "__ffma2_rn"):
        assert name in block, name
    assert "<<<" not in block and "__global__" not in block
    (tmp_path / "wk_acc_extract.inc").write_text(block)
    exe = tmp_path / "wk_acc_harness"
    build = subprocess.run(["g++", "-std=c++17", "-O1", "-ffp-contract=off", f"-I{CUDA_INC}", f"-I{tmp_path}",
                            "-Wno-attributes", "-o", str(exe), str(ROOT / "tests" / "host" / "wk_acc_harness.cpp")],
                           capture_output=True, text=True, timeout=600)
    assert build.returncode == 0, build.stderr[-2000:]
    run = subprocess.run([str(exe)], capture_output=True, text=True, timeout=300)
    assert run.returncode == 0 and run.stdout.startswith("ok "), run.stdout[-2000:] + run.stderr[-2000:]

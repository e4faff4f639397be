"""Host logic of bench.py that needs no GPU: the stamp that ties profiles/ncu_constants.json to the sources."""
import json
from pathlib import Path

import bench

ROOT = Path(bench.__file__).resolve().parent


def test_stamp_ignores_comments_and_sees_code(tmp_path, monkeypatch):
    monkeypatch.setattr(bench, "ROOT", tmp_path)
    (tmp_path / "k.cu").write_text("/* a kernel */\nint f(int x) { return x + 1; }   // plus one\n")
    a = bench.sources_sha1(["k.cu"])
    (tmp_path / "k.cu").write_text("/* reworded\n comment */ int f(int x)\n{\n    return x + 1;\n}\n")
    assert bench.sources_sha1(["k.cu"]) == a
    (tmp_path / "k.cu").write_text("/* a kernel */\nint f(int x) { return x + 2; }\n")
    assert bench.sources_sha1(["k.cu"]) != a


def test_constants_are_withheld_when_the_sources_differ(tmp_path, monkeypatch):
    table = json.loads((ROOT / "profiles" / "ncu_constants.json").read_text())["kernels"]
    assert table, "no captures committed"
    for name, ent in table.items():
        assert (ROOT / ent["capture"]).exists(), ent["capture"]
        for src in ent["sources"]:
            assert (ROOT / src).exists(), src
        for key in ("fma_pipe_active", "dram_bytes_per_launch", "fp32_flops_per_spot", "sources_sha1"):
            assert key in ent, (name, key)
    name, ent = next(iter(table.items()))
    got, note = bench.ncu_constants("no_such_kernel<1>")
    assert got is None and "no ncu capture" in note
    fake = dict(table)
    fake[name] = dict(ent, sources_sha1="0" * 40)
    f = tmp_path / "c.json"
    f.write_text(json.dumps({"kernels": fake}))
    monkeypatch.setattr(bench, "NCU_JSON", f)
    got, note = bench.ncu_constants(name)
    assert got is None and "sources changed" in note

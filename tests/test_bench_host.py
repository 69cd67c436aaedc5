"""Host-side checks of the measurement plumbing (no GPU): the committed ncu stage counters parse and carry a source
hash, the freshness label follows the sources, and `bench.py --impl reference` prints the contract's JSON line."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_committed_stage_counters_parse_and_are_labelled():
    from paper_2607_04230_b200 import ncu_summary
    stages, sha = ncu_summary.read_stage_csv(os.path.join(ROOT, "profiles", "r3_ncu_stage_counters.csv"))
    assert set(stages) == {"generate", "raster", "shade", "filter"}
    for k, d in stages.items():
        assert d["dram_bytes"] > 0 and d["warp_inst"] > 0 and d["duration_ns"] > 0, (k, d)
    assert str(stages["raster"]["kernels"]).count("k_raster") == 2 and "k_hiz" in stages["raster"]["kernels"]
    assert len(sha) == 16 and sha == sha.lower()
    sys.path.insert(0, ROOT)
    import bench
    counters, meta = bench.ncu_counters()
    assert counters["raster"]["warp_inst"] == stages["raster"]["warp_inst"]
    assert meta["fresh"] == (meta["captured_src_sha256"] == ncu_summary.source_hash())
    assert meta["label"].startswith("fresh" if meta["fresh"] else "stale")


def test_source_hash_sees_tokens_but_not_comments(tmp_path, monkeypatch):
    from paper_2607_04230_b200 import ncu_summary
    d = tmp_path / "csrc"
    d.mkdir()
    (d / "a.cu").write_text("__global__ void k(int* p) { p[0] = 1; }  // one\n")
    monkeypatch.setattr(ncu_summary, "CSRC", str(d))
    h0 = ncu_summary.source_hash()
    (d / "a.cu").write_text("/* header */\n__global__ void k(int* p) {\n  p[0] = 1;  // another comment\n}\n")
    assert ncu_summary.source_hash() == h0
    (d / "a.cu").write_text("__global__ void k(int* p) { p[0] = 2; }\n")
    assert ncu_summary.source_hash() != h0


def test_reference_arm_prints_the_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                        "--config", "1"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "Gsegments/s" and line["value"] > 0
    assert line["higher_is_better"] is True and line["vs_baseline"] is None and line["gpu_launches"] == 0
    cb = line["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] == 1 and cb["value"] == line["value"] and cb["cpu_model"]
    assert set(cb["stage_seconds_last_step"]) == {"O1_lod_scan", "O2_generate", "O4_raster_resolve", "O6_shade", "O7_filter"}
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}

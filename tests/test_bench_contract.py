"""bench.py's reference arm (the oracle timed on the host cores) runs without a GPU: its JSON line must carry the keys the
bench contract names, for the workload asked for.  The GPU arm's line is produced on the GPU box (profiles/r2_bench_mw134m.json)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line_with_the_contract_keys():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
                          "--steps", "1", "--warmup", "1"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["higher_is_better"] is True and d["n_gpus"] == 1
    assert d["steps"] == 1 and d["warmup"] == 1 and d["ms_per_step"] > 0 and d["value"] > 0
    assert d["unit"] == "interactions/s" and d["metric"].startswith("tree-force interactions/s")
    assert d["config"]["workload"] == "plummer_16k" and d["vs_baseline"] is None and d["data"] == "synthetic"
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == d["value"] and cb["sample"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["gpu_launches"] == 0


def test_gpu_arm_line_of_round_2_carries_roofline_cpu_baseline_and_e2e():
    d = json.loads(open(os.path.join(ROOT, "profiles", "r2_bench_mw134m.json")).read().strip().splitlines()[-1])
    assert d["config"]["workload"] == "mw_134m" and d["n_gpus"] == 1 and d["dtype"] == "f32"
    r = d["roofline"]
    assert r["bound"] == "alu" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and r["traffic"] > 0
    assert r["kernel_ms_avg"] <= d["ms_per_step"]
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == 16 * d["config"]["n_per_gpu"] == e["d2h_bytes_per_step"] and 0 < e["value"] < d["value"]
    assert d["gpu_launches"] > 0 and d["clocks"]["reasons"] == []
    assert {c["workload"] for c in d["configs"]} == {"plummer_16k", "plummer_1m", "mw_8m", "mw_33m_leapfrog"}

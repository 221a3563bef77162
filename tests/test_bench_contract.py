"""bench.py contract checks that need no GPU: the reference arm (the oracle on the host cores) prints one JSON line with
the agreed keys; the algorithmic-work constants match DESIGN.md section 8."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_the_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0", "--steps", "1",
                        "--warmup", "0"], capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "views/s" and d["higher_is_better"] is True
    assert d["metric"].startswith("candidate views scored/sec") and d["value"] > 0 and d["dtype"] == "f64"
    assert d["config"]["workload"].startswith("BASELINE.json configs[0]") and d["data"] == "synthetic"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "views/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["vs_baseline"] is None and d["n_gpus"] == 1 and d["steps"] == 1


def test_reference_arm_on_other_ranks_is_silent():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0", "--steps", "1",
                        "--warmup", "0", "--gpus", "2"], capture_output=True, text=True, timeout=300, cwd=ROOT, env=env)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_work_constants_match_the_design_document():
    sys.path.insert(0, ROOT)
    import bench
    text = open(os.path.join(ROOT, "DESIGN.md")).read()
    assert bench.FLOP_TEST == 11 and "| 11 flop | `FLOP_TEST` |" in text
    assert bench.FLOP_FWD_PAIR == 31 and "| 31 flop | `FLOP_FWD_PAIR` |" in text
    assert bench.FLOP_BWD_PAIR == {3: 134, 4: 154} and "| 154 (134) flop | `FLOP_BWD_PAIR` |" in text

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


def test_work_constants_come_from_the_committed_counter_pass():
    """roofline.frac uses EXECUTED flop per (pixel, entry) evaluation; the numbers must be the ones of the committed ncu
    metric pass bench.FLOP_SOURCE names (frac must follow from committed counters) and DESIGN.md must quote them"""
    sys.path.insert(0, ROOT)
    import bench
    src = os.path.join(ROOT, bench.FLOP_SOURCE)
    assert os.path.exists(src), bench.FLOP_SOURCE
    prof = open(src).read()
    design = open(os.path.join(ROOT, "DESIGN.md")).read()
    for v in (bench.FLOP_PER_EVAL["forward"], bench.FLOP_PER_EVAL["backward"][3], bench.FLOP_PER_EVAL["backward"][4]):
        assert ("%.1f" % v) in prof, v
        assert ("%.1f" % v) in design, v
    assert "FLOP_PER_EVAL" in design


def test_reference_arm_says_what_it_ran():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0", "--steps", "1",
                        "--warmup", "0"], capture_output=True, text=True, timeout=300, cwd=ROOT)
    d = json.loads(r.stdout.strip().splitlines()[-1])
    assert d["config"]["candidates_per_step"] == 4 and d["config"]["training_views"] == 1
    assert d["config"]["workload_candidates"] == 4 and d["config"]["workload_training_views"] == 1
    assert "cpu" in d["cpu_baseline"]

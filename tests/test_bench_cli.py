"""bench.py's reference arm (`--impl reference`: the fp64 oracle on the host cores) through its command line - CPU only.
The arm of the library itself needs a GPU and is exercised by the driver; here the contract's JSON line is checked on
the small config, and that ranks other than 0 of a torchrun launch print nothing and exit 0."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(extra_env=None):
    env = dict(os.environ, **(extra_env or {}))
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1", "--steps", "2",
           "--warmup", "1"]
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=300)


def test_reference_arm_prints_one_contract_line():
    r = _run()
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [x for x in r.stdout.splitlines() if x.startswith("{")]
    assert len(lines) == 1
    o = json.loads(lines[0])
    assert o["impl"] == "reference" and o["n_gpus"] == 1 and o["steps"] == 2 and o["warmup"] == 1
    assert o["metric"] == "fwd+pose-grad Gray-steps/s" and o["unit"] == "Gray-steps/s" and o["higher_is_better"] is True
    assert o["dtype"] == "f64" and o["data"] == "synthetic" and o["vs_baseline"] is None and o["gpu_launches"] == 0
    assert o["value"] > 0 and o["ms_per_step"] > 0
    assert "C1" in o["config"]["workload"] and "sample" in o["config"]
    cb = o["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == o["value"] and cb["sample"]
    assert o["e2e"] == {"value": o["value"], "unit": o["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_reference_arm_other_ranks_exit_quietly():
    r = _run({"RANK": "1", "LOCAL_RANK": "1", "WORLD_SIZE": "2"})
    assert r.returncode == 0, r.stderr[-2000:]
    assert not [x for x in r.stdout.splitlines() if x.startswith("{")]

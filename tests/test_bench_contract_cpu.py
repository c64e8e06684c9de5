"""The reference arm of bench.py (this tier: the oracle on the host cores) and the JSON contract of its line,
on CPU.  The GPU arm needs a B200 and is exercised by the driver."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args, env=None):
    e = dict(os.environ)
    e.update(env or {})
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                       env=e, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    return r.stdout.strip().splitlines()


def test_reference_arm_prints_one_contract_line():
    lines = _run("--impl", "reference", "--steps", "1", "--warmup", "0", "--config", "0")
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "particle-updates/s" and d["higher_is_better"] is True
    assert d["metric"].startswith("particle-updates/sec") and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["value"] > 0 and d["n_gpus"] == 1 and d["steps"] == 1 and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == 1
    assert d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"] == "configs[0]"


def test_reference_arm_other_ranks_exit_quietly():
    lines = _run("--impl", "reference", "--steps", "1", "--warmup", "0", "--config", "0",
                 env={"RANK": "1", "WORLD_SIZE": "2", "LOCAL_RANK": "1"})
    assert lines == []


def test_oracle_worker_line():
    lines = _run("--oracle-worker", "--config", "0", "--oracle-budget", "0.5")
    d = json.loads(lines[-1])
    assert d["kind"] == "oracle" and d["cores"] == 1 and d["value"] > 0

"""bench.py's reference arm on CPU (no GPU needed): `--impl reference` times the CPU oracle on a bounded sample and prints ONE
JSON line with the keys of the driver's contract; under torchrun only rank 0 prints. The GPU arm's line is checked for the same
keys by the GPU run itself (tests marked gpu cover the kernels; this file covers the host-side contract)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
KEYS = {"impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
        "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"}


def run(env_extra=None):
    env = dict(os.environ, **(env_extra or {}))
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "tiny",
                        "--steps", "2", "--warmup", "1"], capture_output=True, text=True, env=env, timeout=600, cwd=ROOT)
    assert p.returncode == 0, p.stderr[-2000:]
    return p.stdout


def test_reference_arm_prints_one_contract_line():
    out = [l for l in run().splitlines() if l.strip()]
    assert len(out) == 1
    line = json.loads(out[0])
    assert KEYS <= set(line)
    assert line["impl"] == "reference" and line["dtype"] == "f64" and line["data"] == "synthetic"
    assert line["steps"] == 2 and line["warmup"] == 1 and line["higher_is_better"] is True and line["vs_baseline"] is None
    assert line["value"] > 0 and line["ms_per_step"] > 0 and line["unit"] == "tokens/s"
    assert line["config"]["workload"] == "tiny" and "model" not in line["config"]
    cb = line["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == line["value"] and "sample" in cb
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_reference_arm_other_ranks_print_nothing():
    assert run({"RANK": "1", "WORLD_SIZE": "2", "LOCAL_RANK": "1"}).strip() == ""

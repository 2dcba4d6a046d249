"""The bench.py contract that can be checked without a GPU: the reference arm (`--impl reference`: the oracle as it stands on
the host cores, bounded sample) prints ONE JSON line with the keys the driver reads, for the EM path and for both thermal
placements; under a multi-rank launch only rank 0 prints; the default arm refuses to run without a CUDA device (no fallback)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(args, env=None, timeout=600):
    e = dict(os.environ); e.update(env or {})
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, capture_output=True, text=True, cwd=ROOT, env=e, timeout=timeout)


@pytest.mark.parametrize("extra", [[], ["--thermal"], ["--thermal-nodal"]], ids=["em", "thermal-cell", "thermal-node"])
def test_reference_arm_prints_the_contract_line(extra):
    r = _run(["--impl", "reference", "--config", "6", "--steps", "2", "--warmup", "1"] + extra)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "EM cell-updates/sec" and d["unit"] == "cell-updates/s"
    assert d["higher_is_better"] is True and d["n_gpus"] == 1 and d["steps"] == 2 and d["warmup"] == 1
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["vs_baseline"] is None and d["data"] == "synthetic"
    assert "workload" in d["config"] and "model" not in d["config"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == d["value"] and cb["sample"]
    assert d["e2e"]["value"] == d["value"] and d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0


def test_reference_arm_other_ranks_stay_silent():
    r = _run(["--impl", "reference", "--config", "6", "--steps", "1", "--warmup", "1", "--gpus", "2"],
             env={"RANK": "1", "LOCAL_RANK": "1", "WORLD_SIZE": "2", "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": "29999"})
    assert r.returncode == 0 and not [l for l in r.stdout.splitlines() if l.startswith("{")]


def test_default_arm_has_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    r = _run(["--config", "1", "--steps", "1", "--warmup", "3", "--no-cpu-baseline", "--no-e2e"])
    assert r.returncode != 0
    assert not [l for l in r.stdout.splitlines() if l.startswith("{") and "value" in l]

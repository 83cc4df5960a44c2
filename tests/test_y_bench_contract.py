"""bench.py prints ONE JSON line with the keys the round-end driver reads.  Here: the reference arm (`--impl reference`, the
oracle on host cores: no GPU needed) on configs[0], and that every rank but 0 stays silent under torchrun's environment;
the GPU arm's line is checked by the test marked gpu (configs[0], a second-long run)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
             "vs_baseline", "dtype", "data", "config", "e2e")


def _run(args, env=None, timeout=600):
    e = dict(os.environ)
    e.update(env or {})
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, cwd=ROOT, env=e, capture_output=True, text=True,
                       timeout=timeout)
    assert p.returncode == 0, p.stderr[-2000:]
    return [ln for ln in p.stdout.splitlines() if ln.strip()]


def _check_common(d, steps):
    for k in BASE_KEYS:
        assert k in d, k
    assert d["unit"] == "transitions/s" and d["higher_is_better"] is True and d["scaling"] == "weak"
    assert d["steps"] == steps and d["n_gpus"] == 1 and d["data"] == "synthetic"
    assert d["value"] > 0 and d["ms_per_step"] > 0
    assert d["vs_baseline"] is None            # BASELINE.md holds no number of the paper for this metric and workload
    assert "workload" in d["config"] and "model" not in d["config"]
    assert d["dtype"].startswith("f64")
    for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"):
        assert k in d["e2e"], k


def test_reference_arm_line_and_silent_ranks():
    lines = _run(["--impl", "reference", "--config", "0", "--steps", "1", "--warmup", "0", "--ref-seconds", "1"])
    assert len(lines) == 1
    d = json.loads(lines[0])
    _check_common(d, 1)
    assert d["impl"] == "reference"
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["sample"] and cb["value"] == d["value"]
    assert d["e2e"]["value"] == d["value"] and d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["config"]["workload"].startswith("configs[0]")
    # under torchrun every rank but 0 exits 0 without work or output
    assert _run(["--impl", "reference", "--config", "0", "--steps", "1", "--warmup", "0"],
                env={"RANK": "1", "LOCAL_RANK": "1", "WORLD_SIZE": "2"}) == []


@pytest.mark.gpu
def test_gpu_arm_line():
    lines = _run(["--config", "0", "--steps", "2", "--warmup", "1", "--no-cpu-baseline", "--no-per-config"])
    assert len(lines) == 1
    d = json.loads(lines[0])
    _check_common(d, 2)
    assert "impl" not in d or d["impl"] != "reference"
    assert d["warmup"] >= 3 and d.get("warmup_requested") == 1     # the timing rule: at least three untimed steps
    assert d["gpu_launches"] > 0
    r = d["roofline"]
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert k in r, k
    assert r["bound"] == "tensor" and r["unit"] == "TFLOP/s" and r["kernel"] == "rank_k3m_kernel"
    assert abs(r["frac"] - r["achieved"] / r["peak"]) <= 1e-9 * r["frac"]
    c = d["clocks"]
    assert "sm_mhz" in c and "sm_max_mhz" in c and isinstance(c["reasons"], list)
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
    assert d["e2e"]["value"] != d["value"]
    assert d["rank_k_i8"]["mode"].startswith("rpa_chi0_set_rank_k_mode") or "note" in d["rank_k_i8"]

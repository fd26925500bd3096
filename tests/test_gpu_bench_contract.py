"""bench.py's output contract on a GPU box: one JSON line with the keys the driver reads, for both arms and for the
fit mode, on event counts small enough to finish in seconds (the --mc / --data overrides change sizes only)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                         cwd=ROOT, timeout=900)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout[-2000:]
    return json.loads(lines[0])


def test_ours_line_has_the_contract_keys():
    d = _run("--gpus", "1", "--steps", "3", "--warmup", "3", "--mc", "200000", "--data", "20000", "--ref-events", "200000")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks"):
        assert k in d, k
    assert d["metric"] == "nll_grad_hvp_events_per_s" and d["unit"] == "events/s" and d["dtype"] == "f64"
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] >= 3 and d["higher_is_better"] is True
    assert d["vs_baseline"] is None and d["data"] == "synthetic" and "workload" in d["config"]
    rl = d["roofline"]
    assert rl["bound"] == "hbm" and rl["unit"] == "GB/s" and rl["peak"] > 1000 and 0 < rl["frac"] < 1.2
    assert abs(rl["frac"] - rl["achieved"] / rl["peak"]) < 1e-12 and rl["launches_timed"] == 3
    assert d["gpu_launches"] == 2 * 3  # sweep + reduction per step
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] > 0 and "sample" in cb
    assert cb["nll_rel_diff_vs_gpu"] is not None and cb["nll_rel_diff_vs_gpu"] < 1e-10
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == 2 * 120 * 8 and e["d2h_bytes_per_step"] == (1 + 2 * 120) * 8
    assert e["value"] <= d["value"] * 1.05
    assert d["value"] > 100 * cb["value"]  # a GPU sweep, not a CPU fallback


def test_reference_line():
    d = _run("--impl", "reference", "--gpus", "1", "--steps", "2", "--warmup", "1", "--ref-events", "100000")
    assert d["impl"] == "reference" and d["metric"] == "nll_grad_hvp_events_per_s" and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_fit_mode_line():
    d = _run("--config", "5", "--fits", "3", "--mc", "50000", "--data", "5000")
    assert d["metric"] == "fit_seconds" and d["higher_is_better"] is False and len(d["fits"]) == 3
    # round 1 saw this fit stop unconverged (status 5): a width sat on gamma_max and every Armijo trial beyond it halved t
    # to zero (PWA_FIT_TRACE: 20 infeasible trials, |g|inf 25).  The projected Newton-CG of DESIGN.md S15' ends it properly.
    assert d["fit_from_theta_true"]["status"] == 0 and d["fit_from_theta_true"]["nll"] < 0.0
    assert all(r["status"] in (0, 5) and r["sweeps"] > 0 for r in d["fits"])
    if "best" in d:
        b = d["best"]
        assert abs(b["nll"] - b["oracle_nll_at_best_theta"]) <= 1e-9 * abs(b["nll"])


def test_shape_and_store_flags():
    """--shape (another model shape on the config's recipe) and --store copy (library-owned copy; tiled for shapes that
    need 8-event tiles): same contract line, no stored traffic figure for a non-BASELINE shape."""
    d = _run("--shape", "40,4,3", "--mc", "60000", "--data", "6000", "--store", "copy", "--steps", "3", "--warmup", "3",
             "--no-cpu-baseline", "--sustained-seconds", "0")
    assert "shape 40,4,3" in d["config"]["workload"] and "R=40 H=4 C=3" in d["config"]["workload"]
    assert d["config"]["store"] == "library-owned copy" and "tile=8t," in d["config"]["kernel_variant"]
    assert d["roofline"]["traffic"] is None and d["roofline"]["bytes_per_launch"] == 66000 * (16 * 40 * 4 + 8 * 3) + 6000 * 8
    assert d["clocks"]["sm_mhz"] is not None

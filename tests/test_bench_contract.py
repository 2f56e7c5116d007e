"""bench.py prints ONE JSON line with the keys the driver reads (both arms)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step",
             "higher_is_better", "scaling", "vs_baseline", "dtype", "data", "config", "e2e",
             "gpu_launches"}


def _run(*args, timeout=600):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + list(args),
                         capture_output=True, text=True, timeout=timeout, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, out.stdout
    return json.loads(lines[0])


def test_reference_arm_times_the_oracle_on_cpu():
    d = _run("--impl", "reference", "--steps", "1", "--warmup", "1", "--ref-particles", "16")
    assert BASE_KEYS <= set(d)
    assert d["impl"] == "reference" and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == 1
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0,
                        "d2h_bytes_per_step": 0}
    assert d["value"] > 1e6          # > 1e6 particle-steps/s on one core


@pytest.mark.gpu
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_gpu_arm_json_line(prec):
    d = _run("--steps", "3", "--warmup", "3", "--no-extras", "--precision", prec)
    assert BASE_KEYS | {"roofline", "clocks", "forward_ms"} <= set(d)
    assert d["dtype"] == prec and d["n_gpus"] == 1 and d["steps"] == 3
    # build_stream, pack_key, pack_gather, queue init, integrate, pack_scatter, best,
    # gbest, move
    assert d["gpu_launches"] == 3 * 9
    r = d["roofline"]
    assert r["bound"] == "alu" and 0.05 < r["frac"] < 1.0
    assert r["achieved"] == pytest.approx(r["frac"] * r["peak"])
    # the kernel alone (library-recorded events) is shorter than the whole forward call
    assert 0.5 * d["forward_ms"] < r["kernel_ms"] < d["forward_ms"] < d["ms_per_step"]
    # ncu figures come from the committed summary and only while it matches the source
    n = r["ncu"]
    if n["status"] == "fresh":
        assert r["traffic"] > 0 and 0.0 < r["frac_pipe_elapsed"] <= r["frac_pipe_active"] < 1.0
        assert ("integrate_misfit_%s" % prec) in n["kernel"]
    else:
        assert r["traffic"] is None and r["frac_pipe_active"] is None
    e = d["e2e"]
    state = 65536 * 8 * (3 * 2 + 1) + 8 * (2 + 1)       # x, v, pbest, pbestJ, gbest, gbestJ
    assert e["d2h_bytes_per_step"] == 65536 * 8 + state
    assert e["h2d_bytes_per_step"] > 2_000_000 + state
    assert 0.5 * d["value"] < e["value"] <= 1.05 * d["value"]
    assert d["config"]["workload"].startswith("configs[1]")
    assert d["value"] > 5e10

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


def _free_port():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("mode", ["particles", "traces"])
def test_sharded_flag_partitions_as_design_says_world2(mode):
    """bench.py --sharded ... --plan-only under a 2-rank gloo group (no GPU): the
    flag parses and the partition is DESIGN.md section 9's: configs[3]'s 8 192
    particles cut into two contiguous slices with one collective of D + 2 doubles
    per rank and batch; configs[4]'s 256 pixels dealt 128 + 128 with none."""
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen(
            [sys.executable, os.path.join(ROOT, "bench.py"), "--sharded", mode, "--plan-only",
             "--gpus", "2"], env=env, cwd=ROOT, stdout=subprocess.PIPE,
            stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    assert outs[1][0].strip() == ""                      # only rank 0 prints
    d = json.loads(outs[0][0].strip())
    assert d["n_ranks"] == 2 and d["sharded"] == mode
    a, b = d["plan"]
    if mode == "particles":
        assert d["workload"] == "configs[3]"
        assert (a["first_particle"], a["particles_per_trace"]) == (0, 4096)
        assert (b["first_particle"], b["particles_per_trace"]) == (4096, 4096)
        assert a["n_traces"] == b["n_traces"] == 1
        assert a["collective_per_batch"] and a["row_doubles"] == 4 + 2
    else:
        assert d["workload"] == "configs[4]"
        assert (a["n_traces"], b["n_traces"]) == (128, 128)
        assert (a["first_particle"], b["first_particle"]) == (0, 128 * 4096)
        assert a["particles_per_trace"] == b["particles_per_trace"] == 4096
        assert not a["collective_per_batch"] and a["row_doubles"] == 0


@pytest.mark.gpu
@pytest.mark.parametrize("mode", ["particles", "traces"])
def test_sharded_arm_runs_on_one_gpu(mode):
    """The sharded arm itself (world size 1: no process group), a few batches."""
    d = _run("--sharded", mode, "--sharded-iters", "3")
    assert BASE_KEYS <= set(d) and d["scaling"] == "strong" and d["n_gpus"] == 1
    assert d["inversion_ms"] > 0 and d["gpu_launches"] > 0
    assert d["config"]["workload"].startswith("configs[%d]" % (3 if mode == "particles" else 4))


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

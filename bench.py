#!/usr/bin/env python
"""bench.py -- RK4 particle-steps/s of the dAFM force-inversion hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--precision f64|f32] [--no-extras]

Workload (config.workload): BASELINE.json configs[1] -- 65,536 DMT parameter sets,
200 cycles x 256 RK4 steps, random initial phases, misfit over the last 100
cycles against a 25,600-sample noisy trace.  One "step" is one pass of the whole
hot path over that batch: afm_forward_batch (a1-a4: parameter map, RK4, misfit)
followed by afm_pso_step (a5-a7: personal best, global best, Eq. 8 move) on a
65,536-particle swarm holding the same coordinates.  Inputs are synthetic
(paper_1109_0334_b200.workloads, seeded), resident in HBM for `value`, and
start in pinned host memory for `e2e` (afm_forward_batch_host +
afm_pso_step_host: H2D of theta, z0v0, the trace, the misfits and the swarm
state, D2H of the misfits and the swarm state, inside the timed region).

N > 1 (torchrun): every rank runs its own batch of the same shape (different
seeds); there is no data-path collective; scaling is
weak; value = all ranks' particle-steps / max-over-ranks time.

--impl reference times the CPU oracle (oracle/, single thread) on a bounded
sample of the same workload.

--sharded particles|traces (with torchrun for N > 1) runs ONE inversion sharded over
the ranks with paper_1109_0334_b200.sharded.ShardedSwarm: configs[3] cut by particles
(one NCCL all-gather of a candidate row per rank and batch) or configs[4] dealt by
pixels (no collective in the loop); strong scaling; see run_sharded.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1109_0334_b200 import workloads as wlm  # noqa: E402

METRIC = "rk4_particle_steps_per_sec"
UNIT = "particle-steps/s"

# Algorithmic flops per particle-step, SURVEY.md 8(d) / DESIGN.md "Roofline":
# oracle-form arithmetic, add/mul/compare = 1, FMA = 2, div = sqrt = exp = 1.
FLOPS_PER_STEP = {wlm.LAW_DMT: 57.0, wlm.LAW_DMT_VISC: 57.0, wlm.LAW_LJ_EXP: 93.0,
                  wlm.LAW_NONE: 49.0}
# FP64 FMA peak of the lane model: 148 SMs x 64 lanes x 2 flops x clock
N_SM, FP64_LANES, FP32_LANES = 148, 64, 128
# ncu figures of the dominant kernel (DRAM traffic per launch, pipe utilisation) are
# read from the machine-written summary profiles/<PROFILE>_ncu.csv (key,value rows
# taken from `ncu -i <report> --page raw --csv`, with the hash of the library source
# the report belongs to) and reported only while the library source is the one that
# summary was made from; otherwise they are null.
PROFILE = {"f64": "r3_cfg1_f64", "f32": "r3_cfg1_f32"}
PIPE_METRIC = {"f64": "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_",
               "f32": "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_"}


def _ncu_profile(precision):
    """dict(traffic, pipe_active_pct, pipe_elapsed_pct, ...) from the committed ncu
    summary of this precision's integrate kernel, or the reason it is not usable."""
    import csv
    from paper_1109_0334_b200 import build as afm_build
    path = os.path.join(ROOT, "profiles", PROFILE[precision] + "_ncu.csv")
    out = {"file": os.path.relpath(path, ROOT), "traffic": None, "pipe_active_pct": None,
           "pipe_elapsed_pct": None}
    if not os.path.exists(path):
        out["status"] = "no summary committed"
        return out
    kv = dict((r[0], r[1]) for r in csv.reader(open(path)) if len(r) == 2)
    out["kernel"] = kv.get("kernel", "").split("(")[0]
    out["registers_per_thread"] = kv.get("launch__registers_per_thread")
    sha = afm_build.source_sha()
    if kv.get("source_sha") != sha:
        out["status"] = "stale: summary made from source %s, running %s" % (
            kv.get("source_sha"), sha)
        return out
    if ("integrate_misfit_%s" % precision) not in out["kernel"]:
        out["status"] = "summary is of another kernel"
        return out
    out["status"] = "fresh"
    out["traffic"] = int(float(kv["dram_bytes_read"]) + float(kv["dram_bytes_write"]))
    out["pipe_active_pct"] = float(kv[PIPE_METRIC[precision] + "active"])
    out["pipe_elapsed_pct"] = float(kv[PIPE_METRIC[precision] + "elapsed"])
    out["kernel_ms_under_ncu"] = float(kv["duration_ms"])
    key = "fp32" if precision == "f32" else "fp64"
    if ("executed_%s_fma" % key) in kv:
        # warp-instructions x 32 lanes; FMA = 2 flops (SURVEY.md 8(d) definition (2))
        out["executed_flops_per_launch"] = 32.0 * (
            2.0 * float(kv["executed_%s_fma" % key]) + float(kv["executed_%s_add" % key])
            + float(kv["executed_%s_mul" % key]))
    return out


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    sm_max = 1965.0
    src = "fallback clock 1965 MHz"
    if os.path.exists(path):
        try:
            sm_max = float(json.load(open(path)).get("sm_max_mhz", sm_max))
            src = "MEASURED_PEAKS.json sm_max_mhz"
        except Exception:
            pass
    return dict(fp64_tflops=N_SM * FP64_LANES * 2 * sm_max * 1e6 / 1e12,
                fp32_tflops=N_SM * FP32_LANES * 2 * sm_max * 1e6 / 1e12,
                clock_mhz=sm_max, clock_source=src)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
                pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return dict(sm_mhz=float(np.median(sm)) if sm else None,
                    sm_max_mhz=float(max(mx)) if mx else None,
                    power_w_max=float(max(pw)) if pw else None,
                    samples=len(sm), reasons=sorted(reasons))


def _oracle_trace(wl):
    """The oracle's own trace (no oracle input ever comes from the CUDA path)."""
    from oracle import binding as orc
    bad, win = orc.window(orc.model_from(wl), wl["truth"], wl["z0"], wl["v0"])
    return win[None, :] + wlm.trace_noise(wl, n_traces=1)


def _oracle_sample(wl, n_sample, seed_params, seed_states, trace):
    """Time the oracle as it stands (single thread) on n_sample particles."""
    from oracle import binding as orc
    M = orc.model_from(wl)
    params = wlm.draw_params(wl, n_sample, seed=seed_params)
    z0v0 = wlm.draw_initial_states(wl, n_sample, seed=seed_states)
    t0 = time.perf_counter()
    J = orc.forward_batch(M, params, trace, z0v0=z0v0, openmp=False)
    dt = time.perf_counter() - t0
    return dt, J


def _make_trace(wl):
    """The measured trace of the GPU arm: built by the GPU path itself from the
    ground truth + seeded noise (afm_trajectory); nothing here touches oracle/."""
    from paper_1109_0334_b200 import afm
    zs, _ = afm.afm_trajectory(wl["truth"], afm.cfg_from(wl, n_traces=1), wl["z0"], wl["v0"])
    clean = zs[-wl["n_window"]:]
    return clean[None, :] + wlm.trace_noise(wl, n_traces=1)


def run_reference(args):
    """--impl reference: the CPU oracle on a bounded sample of configs[1]."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import binding as orc
    wl = wlm.config(1)
    trace = _oracle_trace(wl)
    n_sample = args.ref_particles
    for _ in range(args.warmup):
        _oracle_sample(wl, 4, 1, 2, trace)
    times = []
    for _ in range(args.steps):
        dt, _ = _oracle_sample(wl, n_sample, 1, 2, trace)
        times.append(dt)
    total = float(sum(times))
    value = n_sample * wl["n_steps"] * args.steps / total
    sample = "%d of 65536 particles x %d RK4 steps per step, single thread" % (
        n_sample, wl["n_steps"])
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[1] forward batch, DMT, FP64 (bounded sample)",
                   "particles_per_step": n_sample, "rk4_steps": wl["n_steps"]},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": sample, "host_cores": os.cpu_count()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0,
                "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))
    return 0


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1109_0334_b200 import afm

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    afm.lib()
    prec = afm.F32 if args.precision == "f32" else afm.F64

    wl = wlm.config(1)
    P = wl["swarm"]["n_particles"]
    D = wl["n_params"]
    N = wl["n_steps"]
    cfg = afm.cfg_from(wl, precision=prec)
    trace_np = _make_trace(wl)
    coords_np = wlm.draw_coords(wl, P, seed=1 + 100 * rank)
    params_np = wlm.theta_of_coords(wl, coords_np)
    z0v0_np = wlm.draw_initial_states(wl, P, seed=2 + 100 * rank)

    dev = torch.device("cuda", local)
    params = torch.as_tensor(params_np, device=dev)
    trace = torch.as_tensor(trace_np, device=dev)
    z0v0 = torch.as_tensor(z0v0_np, device=dev)
    misfit = torch.empty(P, dtype=torch.float64, device=dev)
    bounds = afm.bounds_from(wl)
    swarm = afm.swarm_from(wl)
    state = afm.afm_pso_init(bounds, swarm, D, 1, wl["pso_seed"])
    state["x"].copy_(torch.as_tensor(coords_np, device=dev))
    state["pbest"].copy_(state["x"])
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def step(it):
        afm.afm_forward_batch(params, trace, cfg, z0v0=z0v0, misfit=misfit)
        afm.afm_pso_step(bounds, swarm, D, 1, wl["pso_seed"], it, True, misfit, state)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(args.warmup):
        step(i)
    barrier()

    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True),
           torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    afm.afm_reset_launch_count()
    # the library brackets every integrate-kernel launch with its own event pair
    # on the launching stream: roofline.kernel_ms is that kernel alone
    afm.afm_set_option("kernel_events", 1)
    barrier()
    for i in range(args.steps):
        flush.zero_()                      # L2 flush between timed iterations (untimed)
        ev[i][0].record()
        afm.afm_forward_batch(params, trace, cfg, z0v0=z0v0, misfit=misfit)
        ev[i][1].record()
        afm.afm_pso_step(bounds, swarm, D, 1, wl["pso_seed"], args.warmup + i, True,
                         misfit, state)
        ev[i][2].record()
    barrier()
    launches = afm.afm_launch_count()
    kernel_times = afm.afm_kernel_times(min(args.steps, 64))
    kernel_name = afm.afm_last_integrate_kernel()   # which form the library chose to run
    afm.afm_set_option("kernel_events", 0)
    step_ms = [e[0].elapsed_time(e[2]) for e in ev]
    fwd_ms = [e[0].elapsed_time(e[1]) for e in ev]
    total_ms = float(sum(step_ms))
    clocks = sampler.stop() if sampler else None

    # ---- e2e: the same step through the C ABI with HOST buffers: theta, z0v0, the
    # trace, the misfits and the whole swarm state start and end in (pinned) host
    # memory; every copy is inside the timed region -------------------------------
    def pinned(a):
        return torch.as_tensor(np.ascontiguousarray(a)).pin_memory().numpy()
    hp, ht, hz = pinned(params_np), pinned(trace_np), pinned(z0v0_np)
    ho = pinned(np.empty(P))
    hst = {k: pinned(v.cpu().numpy()) for k, v in state.items()}

    def e2e_step(it):
        afm.afm_forward_batch_host(hp, ht, cfg, z0v0=hz, misfit=ho)
        afm.afm_pso_step_host(bounds, swarm, D, 1, wl["pso_seed"], it, True, ho, hst)

    e2e_step(0)
    barrier()
    t0 = time.perf_counter()
    for i in range(args.steps):
        e2e_step(1 + i)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    finite = int(np.isfinite(ho).sum())
    state_bytes = int(sum(v.nbytes for v in hst.values()))

    t = torch.tensor([total_ms, e2e_s * 1e3, float(sum(fwd_ms))], dtype=torch.float64,
                     device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms, e2e_ms, fwd_total_ms = [float(x) for x in t.cpu()]

    units = float(P) * N * args.steps * world
    value = units / (total_ms * 1e-3)
    e2e_value = units / (e2e_ms * 1e-3)

    if rank == 0:
        pk = _peaks()
        kern_ms = float(np.mean(kernel_times))
        flops = FLOPS_PER_STEP[wl["law"]] * P * N
        achieved = flops / (kern_ms * 1e-3) / 1e12
        peak = pk["fp32_tflops"] if prec == afm.F32 else pk["fp64_tflops"]
        peak_meas = afm.afm_fma_peak(prec, 0.25)
        ncu = _ncu_profile(args.precision)
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if prec == afm.F32 else "f64", "data": "synthetic",
            "config": {"workload": "configs[1]: 65536 DMT theta x 200 cycles x 256 RK4 "
                                   "steps, misfit over last 100 cycles (per GPU)",
                       "particles_per_gpu": P, "rk4_steps": N, "window": wl["n_window"],
                       "step": "afm_forward_batch (warp packing, segment queue) + "
                               "afm_pso_step",
                       "l2": "256 MB buffer zeroed between timed iterations"},
            "e2e": {"value": e2e_value, "unit": UNIT,
                    "h2d_bytes_per_step": int(hp.nbytes + ht.nbytes + hz.nbytes + ho.nbytes
                                              + state_bytes),
                    "d2h_bytes_per_step": int(ho.nbytes + state_bytes),
                    "api": "afm_forward_batch_host + afm_pso_step_host",
                    "finite_misfits": finite},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "forward_ms": fwd_total_ms / args.steps,
            "roofline": {"bound": "alu",
                         "kernel": kernel_name,
                         "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                         "frac": achieved / peak,
                         "kernel_ms": kern_ms,
                         "kernel_ms_source": "CUDA events recorded by the library around "
                                             "each launch of that kernel alone (the queue "
                                             "reset kernel comes before the start event) on "
                                             "its stream, mean of %d timed launches"
                                             % len(kernel_times),
                         "flops_per_particle_step": FLOPS_PER_STEP[wl["law"]],
                         "algorithmic_bytes": int(P * (8 * D + 16 + 8) + N * 32),
                         "traffic": ncu["traffic"],
                         "frac_pipe_active": (None if ncu["pipe_active_pct"] is None
                                              else ncu["pipe_active_pct"] / 100.0),
                         "frac_pipe_elapsed": (None if ncu["pipe_elapsed_pct"] is None
                                               else ncu["pipe_elapsed_pct"] / 100.0),
                         "executed_tflops": (
                             None if not ncu.get("executed_flops_per_launch") else
                             ncu["executed_flops_per_launch"] / (kern_ms * 1e-3) / 1e12),
                         "frac_executed": (
                             None if not ncu.get("executed_flops_per_launch") else
                             ncu["executed_flops_per_launch"] / (kern_ms * 1e-3) / 1e12 / peak),
                         "ncu": ncu,
                         "peak_source": "lane model 148 SM x %d lanes x 2 x %s (%s)" % (
                             FP32_LANES if prec == afm.F32 else FP64_LANES,
                             pk["clock_mhz"], pk["clock_source"]),
                         "peak_measured": peak_meas,
                         "frac_of_measured": achieved / peak_meas,
                         "peak_measured_source": "afm_fma_peak: register-only FMA "
                                                 "chains, 0.25 s, this run"},
        }
        if not args.no_extras and world == 1:
            out["extras"] = extras(afm, torch, dev, prec)
            n_s = args.cpu_particles
            dt, _ = _oracle_sample(wl, n_s, 1, 2, _oracle_trace(wl))
            out["cpu_baseline"] = {
                "value": n_s * N / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                "sample": "%d of 65536 particles x %d RK4 steps, single thread, %.1f s"
                          % (n_s, N, dt),
                "host_cores": os.cpu_count()}
            out["north_star_targets"] = _targets(out, ncu, args.precision)
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def _targets(out, ncu, precision):
    """BASELINE.json:north_star's three targets as plain pass/fail (None: not
    measured by this run)."""
    ex = out.get("extras", {})
    other = _ncu_profile("f32" if precision == "f64" else "f64")
    by = {precision: ncu, ("f32" if precision == "f64" else "f64"): other}

    def pipe(p, bar):
        v = by[p]["pipe_active_pct"]
        return {"pipe_active_pct": v, "pipe_elapsed_pct": by[p]["pipe_elapsed_pct"],
                "bar_pct": bar, "met": None if v is None else bool(v >= bar),
                "source": "builder capture: ncu summary %s committed by the builder, not "
                          "measured by this run" % by[p]["file"],
                "status": by[p]["status"]}
    ms = ex.get("cfg2_inversion_ms")
    return {"fp64_pipe_ge_60pct_configs1": pipe("f64", 60.0),
            "fp32_pipe_ge_50pct_configs1": pipe("f32", 50.0),
            "configs2_inversion_lt_100ms": {"ms": ms, "met": None if ms is None
                                            else bool(ms < 100.0),
                                            "source": "this run (extras.cfg2_inversion_ms)"}}


def _event_ms(torch, fn, reps):
    fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def _wall_ms(fn, warmups, runs):
    """Host wall clock, call to return: `warmups` untimed calls, then the median and
    the best of `runs` timed ones (SURVEY.md 8(d) "Timing").  Returns (median, best,
    last result)."""
    r = None
    for _ in range(warmups):
        r = fn()
    ts = []
    for _ in range(runs):
        t0 = time.perf_counter()
        r = fn()
        ts.append((time.perf_counter() - t0) * 1e3)
    return float(np.median(ts)), float(min(ts)), r


def extras(afm, torch, dev, main_prec):
    """Secondary figures of BASELINE.json:metric (not the headline): measured FMA
    peaks, configs[1] in the other precision, one forward batch and the full
    inversion of configs[3] and [4] at full size, and the inversion wall time (host
    clock, call to return, median of 5 after 3 warm-ups) of configs[0] and [2]."""
    ex = {"fma_peak_measured_tflops": {"f64": afm.afm_fma_peak(afm.F64, 0.25),
                                       "f32": afm.afm_fma_peak(afm.F32, 0.25)},
          "timing": "inversions: host wall clock, call to return; cfg0/cfg2: 3 warm-ups, "
                    "median of 5; cfg3/cfg4 full inversions: 1 warm-up, median of 3 "
                    "(cfg3 f64: 1 run)"}

    def trace_of(wl, truths=None):
        cfg = afm.cfg_from(wl)
        T = wl["n_traces"]
        tl = [wl["truth"]] if truths is None else truths
        rows = [afm.afm_trajectory(tl[s], cfg, wl["z0"], wl["v0"])[0][-wl["n_window"]:]
                for s in range(T)]
        return torch.as_tensor(np.stack(rows) + wlm.trace_noise(wl), device=dev)

    def rel(r, wl):
        return [float(abs(a - t) / abs(t)) for a, t in zip(r["theta_star"][0], wl["truth"])]

    # configs[1] in the other precision (kernel only, CUDA events)
    wl = wlm.config(1)
    P = wl["swarm"]["n_particles"]
    other = afm.F64 if main_prec == afm.F32 else afm.F32
    params = torch.as_tensor(wlm.draw_params(wl, P, seed=1), device=dev)
    z0v0 = torch.as_tensor(wlm.draw_initial_states(wl, P, seed=2), device=dev)
    tr = trace_of(wl)
    out = torch.empty(P, dtype=torch.float64, device=dev)
    cfg = afm.cfg_from(wl, precision=other)
    afm.afm_set_option("kernel_events", 1)
    ms = _event_ms(torch, lambda: afm.afm_forward_batch(params, tr, cfg, z0v0=z0v0,
                                                        misfit=out), 3)
    kt = afm.afm_kernel_times(3)          # the 3 timed launches, the kernel alone
    kname = afm.afm_last_integrate_kernel()
    afm.afm_set_option("kernel_events", 0)
    name = "f64" if other == afm.F64 else "f32"
    ex["cfg1_%s_forward_ms" % name] = ms
    ex["cfg1_%s_particle_steps_per_s" % name] = P * wl["n_steps"] / (ms * 1e-3)
    # the roofline block of the other precision, built like the headline's
    pk = _peaks()
    kms = float(np.mean(kt))
    ach = FLOPS_PER_STEP[wl["law"]] * P * wl["n_steps"] / (kms * 1e-3) / 1e12
    peak = pk["fp64_tflops"] if other == afm.F64 else pk["fp32_tflops"]
    prof = _ncu_profile(name)
    ex["roofline_%s" % name] = {
        "bound": "alu", "kernel": kname, "achieved": ach, "peak": peak, "unit": "TFLOP/s",
        "frac": ach / peak, "kernel_ms": kms,
        "kernel_ms_source": "CUDA events recorded by the library around each launch of "
                            "that kernel alone, mean of %d launches, no L2 flush between "
                            "them" % len(kt),
        "flops_per_particle_step": FLOPS_PER_STEP[wl["law"]],
        "traffic": prof["traffic"],
        "frac_pipe_active": (None if prof["pipe_active_pct"] is None
                             else prof["pipe_active_pct"] / 100.0),
        "frac_pipe_elapsed": (None if prof["pipe_elapsed_pct"] is None
                              else prof["pipe_elapsed_pct"] / 100.0),
        "ncu_source": "builder capture %s (%s)" % (prof["file"], prof["status"]),
        "frac_of_measured": ach / ex["fma_peak_measured_tflops"][name]}

    # configs[3] (both precisions) and configs[4]: one full-size forward batch and the
    # full inversion, measured (not extrapolated)
    for ci, precs in ((3, (afm.F64, afm.F32)), (4, (afm.F64,))):
        wl = wlm.config(ci)
        T, per = wl["n_traces"], wl["swarm"]["n_particles"]
        truths = None if wl["truth"] is not None else wlm.pixel_truths(wl)
        tr = trace_of(wl, truths)
        params = torch.as_tensor(wlm.draw_params(wl, T * per, seed=1), device=dev)
        out = torch.empty(T * per, dtype=torch.float64, device=dev)
        b, sw = afm.bounds_from(wl), afm.swarm_from(wl)
        for prec in precs:
            cfg = afm.cfg_from(wl, precision=prec)
            ms = _event_ms(torch, lambda: afm.afm_forward_batch(params, tr, cfg,
                                                                misfit=out), 2)
            name = "f64" if prec == afm.F64 else "f32"
            ex["cfg%d_%s_batch_ms" % (ci, name)] = ms
            ex["cfg%d_%s_particle_steps_per_s" % (ci, name)] = \
                T * per * wl["n_steps"] / (ms * 1e-3)
            slow = (ci == 3 and prec == afm.F64)
            med, best, r = _wall_ms(lambda: afm.afm_pso_invert(b, sw, wl["pso_seed"], tr, cfg),
                                    0 if slow else 1, 1 if slow else 3)
            ex["cfg%d_%s_full_inversion_s" % (ci, name)] = med * 1e-3
            ex["cfg%d_%s_full_inversion_particle_steps_per_s" % (ci, name)] = \
                float(T) * per * wl["n_steps"] * sw.n_iters / (med * 1e-3)
            if wl["truth"] is not None:
                ex["cfg%d_%s_theta_star_rel_err_vs_truth" % (ci, name)] = rel(r, wl)

    for ci in (0, 2):
        wl = wlm.config(ci)
        cfg = afm.cfg_from(wl)
        trace = trace_of(wl)
        b, s = afm.bounds_from(wl), afm.swarm_from(wl)
        med, best, r = _wall_ms(lambda: afm.afm_pso_invert(b, s, wl["pso_seed"], trace, cfg),
                                3, 5)
        units = wl["swarm"]["n_particles"] * wl["swarm"]["n_iters"] * wl["n_steps"]
        ex["cfg%d_inversion_ms" % ci] = med
        ex["cfg%d_inversion_ms_best" % ci] = best
        ex["cfg%d_particle_steps_per_s" % ci] = units / (med * 1e-3)
        ex["cfg%d_theta_star_rel_err_vs_truth" % ci] = rel(r, wl)
        if ci == 2:
            # the paper's stopping rule is a cost cutoff (DESIGN.md
            # R24); here the cutoff is the noise energy of the trace, W sigma^2 + 3 sd.
            # tests/test_gpu_full_size.py replays this run against the oracle (same
            # number of batches, same theta*).
            W, sg = wl["n_window"], wl["sigma"]
            jt = W * sg * sg * (1.0 + 3.0 * (2.0 / W) ** 0.5)
            sc = afm.swarm_from(wl, j_target=jt)
            med, best, r = _wall_ms(
                lambda: afm.afm_pso_invert(b, sc, wl["pso_seed"], trace, cfg), 3, 5)
            ex["cfg2_time_to_cutoff_ms"] = med
            ex["cfg2_batches_to_cutoff"] = int(r["n_iters_done"])
            ex["cfg2_cutoff_theta_star_rel_err_vs_truth"] = rel(r, wl)
            # the same inversion with a swarm that fills the machine: 1 024 particles
            # are 32 warps on 592 SM sub-partitions, and a batch of 16 384 takes the
            # same time (the time loop is a latency chain), so the swarm can be 16x
            # wider for free and needs far fewer batches.  NOT
            # configs[2] as BASELINE.json states it: another computation, quoted as an
            # observation only.
            for tag, kw in (("to_cutoff", dict(j_target=jt, n_particles=16384)),
                            ("30_batches", dict(n_particles=16384, n_iters=30))):
                sc = afm.swarm_from(wl, **kw)
                med, best, r = _wall_ms(
                    lambda: afm.afm_pso_invert(b, sc, wl["pso_seed"], trace, cfg), 1, 3)
                ex["cfg2_wide16384_%s_ms" % tag] = med
                ex["cfg2_wide16384_%s_batches" % tag] = int(r["n_iters_done"])
                ex["cfg2_wide16384_%s_theta_star_rel_err_vs_truth" % tag] = rel(r, wl)
    return ex


class _PlanBackend:
    """--plan-only: records what ShardedSwarm asks for, computes nothing."""

    def init(self, bounds, swarm, n_dims, n_traces, seed, first):
        import torch
        return {"gbest": torch.zeros((n_traces, n_dims), dtype=torch.float64)}


def run_sharded(args):
    """--sharded particles|traces: ONE inversion sharded over the ranks
    (paper_1109_0334_b200.sharded.ShardedSwarm: CUDA library + NCCL; DESIGN.md
    section 9).  particles: configs[3], one swarm of 8 192 particles cut into
    contiguous slices, one all-gather of a candidate row per rank and batch.  traces:
    configs[4], 256 pixels dealt to the ranks, no collective in the loop.  Total work
    is fixed as N grows: strong scaling.  --plan-only prints the partition of every
    rank and exits (no GPU needed: gloo)."""
    import torch
    import torch.distributed as dist
    from paper_1109_0334_b200.sharded import ShardedSwarm
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    ci = 3 if args.sharded == "particles" else 4
    wl = wlm.config(ci)
    if args.sharded_iters:
        wl = wlm.scaled(wl, n_iters=args.sharded_iters)
    T, per, D = wl["n_traces"], wl["swarm"]["n_particles"], wl["n_params"]

    if args.plan_only:
        from paper_1109_0334_b200 import afm as _afm
        if world > 1:
            dist.init_process_group("gloo")
        cfg, sw = _afm.cfg_from(wl), _afm.swarm_from(wl)
        s = ShardedSwarm(_afm.bounds_from(wl), sw, wl["pso_seed"],
                         torch.zeros((T, wl["n_window"]), dtype=torch.float64), cfg,
                         shard=args.sharded, backend=_PlanBackend())
        mine = {"rank": s.rank, "first_particle": int(s.first),
                "particles_per_trace": int(s.swarm.n_particles), "n_traces": int(s.n_traces),
                "collective_per_batch": bool(s.exchange),
                "row_doubles": _afm.shard_row_doubles(D, sw.topology) if s.exchange else 0}
        plans = [mine]
        if world > 1:
            plans = [None] * world
            dist.all_gather_object(plans, mine)
            dist.destroy_process_group()
        if rank == 0:
            print(json.dumps({"sharded": args.sharded, "workload": "configs[%d]" % ci,
                              "n_ranks": world, "plan": plans}))
        return 0

    if not torch.cuda.is_available():
        raise SystemExit("bench.py --sharded needs CUDA devices: there is no CPU fallback")
    # NCCL's own communicator log (ranks, devices, transports) goes to stderr
    os.environ.setdefault("NCCL_DEBUG", "INFO")
    os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    from paper_1109_0334_b200 import afm
    afm.lib()
    prec = afm.F32 if args.precision == "f32" else afm.F64
    cfg = afm.cfg_from(wl, precision=prec)
    b, sw = afm.bounds_from(wl), afm.swarm_from(wl)
    truths = [wl["truth"]] if wl["truth"] is not None else wlm.pixel_truths(wl)
    c64 = afm.cfg_from(wl)
    rows = [afm.afm_trajectory(truths[s], c64, wl["z0"], wl["v0"])[0][-wl["n_window"]:]
            for s in range(T)]
    h_trace = torch.as_tensor(np.stack(rows) + wlm.trace_noise(wl)).pin_memory()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def one_run(timed):
        trace = h_trace.to(dev, non_blocking=True)            # H2D inside the run
        s = ShardedSwarm(b, sw, wl["pso_seed"], trace, cfg, shard=args.sharded,
                         time_exchange=timed)
        th, Js = s.run()                                      # D2H of theta*, J* inside
        return s, th, Js

    one_run(False)                                            # warm-up
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    afm.afm_reset_launch_count()
    t0 = time.perf_counter()
    s, th, Js = one_run(True)
    barrier()
    wall_ms = (time.perf_counter() - t0) * 1e3
    launches = afm.afm_launch_count()
    clocks = sampler.stop() if sampler else None
    ex = s.exchange_ms()
    t = torch.tensor([wall_ms, float(np.mean(ex)) if ex else 0.0], dtype=torch.float64,
                     device=dev)
    ids = [(rank, torch.cuda.get_device_properties(local).uuid.__str__())]
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        got = [None] * world
        dist.all_gather_object(got, ids[0])
        ids = got
    wall_ms, ex_ms = [float(v) for v in t.cpu()]
    if rank == 0:
        units = float(T) * per * wl["n_steps"] * sw.n_iters
        value = units / (wall_ms * 1e-3)
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": 1,
            "warmup": 1, "ms_per_step": wall_ms, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None,
            "dtype": args.precision, "data": "synthetic",
            "config": {"workload": "configs[%d] inversion sharded by %s over %d rank(s): "
                                   "%d trace(s) x %d particles x %d batches x %d RK4 steps"
                                   % (ci, args.sharded, world, T, per, sw.n_iters,
                                      wl["n_steps"]),
                       "step": "one whole inversion (ShardedSwarm.run)",
                       "collective": ("all_gather of %d doubles per rank and batch (NCCL)"
                                      % afm.shard_row_doubles(D, sw.topology))
                                     if s.exchange else "none in the loop"},
            "inversion_ms": wall_ms,
            "exchange_ms_per_batch": ex_ms if s.exchange else None,
            "theta_star_first": [float(x) for x in th[0]], "J_star_first": float(Js[0]),
            "e2e": {"value": value, "unit": UNIT,
                    "h2d_bytes_per_step": int(h_trace.numel() * 8),
                    "d2h_bytes_per_step": int(th.numel() * 8 + Js.numel() * 8),
                    "api": "ShardedSwarm.run (trace H2D and theta*, J* D2H inside the "
                           "timed region)"},
            "gpu_launches": int(launches), "clocks": clocks,
            "ranks": [{"rank": r, "device_uuid": u} for r, u in ids],
            "nccl_version": ".".join(str(v) for v in torch.cuda.nccl.version())
                            if world > 1 else None}))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def _one_batch_beam(args, afm, torch, dev):
    """--one-batch 7: the paper's 8-mode Euler-Bernoulli forward model
    (workloads.beam_workload): one forward batch of --beam-particles particles, or
    with --invert the 1 024 x 40 inversion."""
    wl = wlm.beam_workload()
    cfg = afm.beam_cfg_from(wl)
    u, _ = afm.afm_beam_trajectory(wl["truth"], cfg)
    trace = torch.as_tensor(u[-wl["n_window"]:][None, :] + wlm.trace_noise(wl), device=dev)
    if args.invert:
        b, sw = afm.bounds_from(wl), afm.swarm_from(wl)
        afm.afm_beam_pso_invert(b, sw, wl["pso_seed"], trace, cfg)
        t0 = time.perf_counter()
        r = afm.afm_beam_pso_invert(b, sw, wl["pso_seed"], trace, cfg)
        ms = (time.perf_counter() - t0) * 1e3
        units = float(sw.n_particles) * wl["n_steps"] * sw.n_iters
        print(json.dumps({"one_batch": 7, "mode": "inversion", "dtype": "f64", "ms": ms,
                          "n_modes": cfg.n_modes,
                          "particle_steps_per_s": units / (ms * 1e-3),
                          "theta_star": [float(x) for x in r["theta_star"][0]]}))
        return 0
    P = args.beam_particles
    params = torch.as_tensor(wlm.draw_params(wl, P, seed=1), device=dev)
    out = torch.empty(P, dtype=torch.float64, device=dev)
    ms = _event_ms(torch, lambda: afm.afm_beam_forward_batch(params, trace, cfg, misfit=out),
                   args.steps)
    # FP64 instructions per particle-step of the 8-mode step
    print(json.dumps({"one_batch": 7, "mode": "forward", "dtype": "f64", "ms": ms,
                      "n_modes": cfg.n_modes, "particles": P,
                      "particle_steps_per_s": float(P) * wl["n_steps"] / (ms * 1e-3),
                      "mode_steps_per_s": float(P) * wl["n_steps"] * cfg.n_modes / (ms * 1e-3)}))
    return 0


def run_one_batch(args):
    """--one-batch CFG: one full-size forward batch (or, with --invert, the full
    inversion) of BASELINE.json configs[CFG], for ncu captures of the other
    launch regimes.  Prints a small JSON line; NOT the bench line."""
    import torch
    from paper_1109_0334_b200 import afm
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    if args.one_batch == 7:
        return _one_batch_beam(args, afm, torch, dev)
    wl = wlm.config(args.one_batch)
    prec = afm.F32 if args.precision == "f32" else afm.F64
    cfg = afm.cfg_from(wl, precision=prec)
    T, per = wl["n_traces"], wl["swarm"]["n_particles"]
    truths = [wl["truth"]] if wl["truth"] is not None else wlm.pixel_truths(wl)
    c64 = afm.cfg_from(wl)
    rows = [afm.afm_trajectory(truths[s], c64, wl["z0"], wl["v0"])[0][-wl["n_window"]:]
            for s in range(T)]
    trace = torch.as_tensor(np.stack(rows) + wlm.trace_noise(wl), device=dev)
    if args.invert:
        b, sw = afm.bounds_from(wl), afm.swarm_from(wl)
        afm.afm_pso_invert(b, sw, wl["pso_seed"], trace, cfg)
        t0 = time.perf_counter()
        r = afm.afm_pso_invert(b, sw, wl["pso_seed"], trace, cfg)
        ms = (time.perf_counter() - t0) * 1e3
        units = float(T) * per * wl["n_steps"] * sw.n_iters
        print(json.dumps({"one_batch": args.one_batch, "mode": "inversion",
                          "dtype": args.precision, "ms": ms,
                          "particle_steps_per_s": units / (ms * 1e-3),
                          "J_star_first": float(r["J_star"][0])}))
        return 0
    params = torch.as_tensor(wlm.draw_params(wl, T * per, seed=1), device=dev)
    z0v0 = (torch.as_tensor(wlm.draw_initial_states(wl, T * per, seed=2), device=dev)
            if args.one_batch == 1 else None)
    out = torch.empty(T * per, dtype=torch.float64, device=dev)
    ms = _event_ms(torch, lambda: afm.afm_forward_batch(params, trace, cfg, z0v0=z0v0,
                                                        misfit=out), args.steps)
    print(json.dumps({"one_batch": args.one_batch, "mode": "forward",
                      "dtype": args.precision, "ms": ms,
                      "particle_steps_per_s": float(T) * per * wl["n_steps"] / (ms * 1e-3)}))
    return 0


def run_pso_step(args):
    """--pso-step CFG: rows a5-a7 of SURVEY.md 8(a) on their own (afm_pso_step:
    pso_best_kernel, pso_gbest_kernel, pso_move_kernel) on a swarm of configs[CFG]'s
    size with seeded synthetic misfits, for ncu captures of the PSO kernels and their
    share of the HBM roofline.  Prints a small JSON line; NOT the bench line."""
    import torch
    from paper_1109_0334_b200 import afm
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    wl = wlm.config(args.pso_step)
    T, per, D = wl["n_traces"], wl["swarm"]["n_particles"], wl["n_params"]
    P = T * per
    b, sw = afm.bounds_from(wl), afm.swarm_from(wl)
    state = afm.afm_pso_init(b, sw, D, T, wl["pso_seed"])
    g = torch.Generator(device=dev)
    g.manual_seed(1234)
    Js = [torch.rand(P, dtype=torch.float64, device=dev, generator=g) for _ in range(4)]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    for i in range(args.warmup):
        afm.afm_pso_step(b, sw, D, T, wl["pso_seed"], i, True, Js[i % 4], state)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(args.steps)]
    afm.afm_reset_launch_count()
    for i in range(args.steps):
        flush.zero_()
        ev[i][0].record()
        afm.afm_pso_step(b, sw, D, T, wl["pso_seed"], args.warmup + i, True, Js[i % 4], state)
        ev[i][1].record()
    torch.cuda.synchronize()
    ms = float(np.mean([a.elapsed_time(z) for a, z in ev]))
    # no-improvement lower bound: best reads J, pbestJ; move reads x, v, pbest and
    # writes x, v (a personal best that improves adds 8 D + 8 bytes read/written)
    algo = 16 * P + 40 * D * P
    hbm = None
    try:
        hbm = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
    except Exception:
        pass
    print(json.dumps({"pso_step": args.pso_step, "particles": P, "n_traces": T, "dims": D,
                      "ms_per_step": ms, "launches_per_step": afm.afm_launch_count() / args.steps,
                      "algorithmic_bytes_per_step": algo,
                      "achieved_gbs": algo / (ms * 1e-3) / 1e9,
                      "hbm_peak_gbs": hbm,
                      "frac": None if not hbm else algo / (ms * 1e-3) / 1e9 / hbm,
                      "l2": "256 MB buffer zeroed between timed steps"}))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"])
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--cpu-particles", type=int, default=3072,
                    help="oracle sample size of the cpu_baseline leg")
    ap.add_argument("--ref-particles", type=int, default=512,
                    help="oracle sample size per step of --impl reference")
    ap.add_argument("--one-batch", type=int, default=None, choices=[0, 1, 2, 3, 4, 7],
                    help="profiling aid: one full-size forward batch of configs[N]; "
                         "7 = the paper's 8-mode beam workload")
    ap.add_argument("--pso-step", type=int, default=None, choices=[0, 1, 2, 3, 4],
                    help="profiling aid: afm_pso_step alone on a swarm of configs[N]'s size")
    ap.add_argument("--beam-particles", type=int, default=65536)
    ap.add_argument("--invert", action="store_true",
                    help="with --one-batch: time the full PSO inversion instead")
    ap.add_argument("--sharded", default=None, choices=["particles", "traces"],
                    help="ONE inversion sharded over the ranks: configs[3] by particles "
                         "(all-gather per batch) or configs[4] by traces (no collective)")
    ap.add_argument("--sharded-iters", type=int, default=0,
                    help="with --sharded: run this many batches instead of the config's")
    ap.add_argument("--plan-only", action="store_true",
                    help="with --sharded: print every rank's partition and exit")
    args = ap.parse_args()
    if args.sharded is not None:
        return run_sharded(args)
    if args.one_batch is not None:
        return run_one_batch(args)
    if args.pso_step is not None:
        return run_pso_step(args)
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())

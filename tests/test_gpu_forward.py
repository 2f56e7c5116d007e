"""GPU parity: afm_forward_batch / afm_trajectory / afm_philox4x32_10 (through the
C ABI) against the CPU oracle on the same seeded inputs.

Tolerance (BASELINE.json:north_star): per-particle misfit within 1e-9 relative
in FP64.  The kernel is not an operation-by-operation copy of the oracle (FMA
contraction, per-step variables, short reciprocal/sqrt sequences), so the two
differ by accumulated rounding: DESIGN.md "Tolerances" derives ~1e-11.
"""
import os

import numpy as np
import pytest

from oracle import binding as orc
from paper_1109_0334_b200 import workloads as wlm
from parity_helpers import oracle_trace, rel_err

pytestmark = pytest.mark.gpu

TOL_F64 = 1e-9
KAT = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


@pytest.fixture(scope="module")
def afm():
    import torch
    assert torch.cuda.is_available()
    from paper_1109_0334_b200 import afm as m
    m.lib()  # fails loudly if the CUDA library is missing
    yield m
    m.afm_set_option("block", 0)
    m.afm_set_option("tile", 0)


def _gpu_forward(afm, wl, params, trace, z0v0=None, **cfg_over):
    import torch
    cfg = afm.cfg_from(wl, **cfg_over)
    p = torch.as_tensor(np.ascontiguousarray(params), device="cuda")
    t = torch.as_tensor(np.ascontiguousarray(trace), device="cuda")
    zv = None if z0v0 is None else torch.as_tensor(np.ascontiguousarray(z0v0), device="cuda")
    J = afm.afm_forward_batch(p, t, cfg, z0v0=zv)
    torch.cuda.synchronize()
    return J.cpu().numpy()


def _oracle_forward(wl, params, trace, z0v0=None):
    return orc.forward_batch(orc.model_from(wl), params, trace, z0v0=z0v0,
                             z0=wl["z0"], v0=wl["v0"], n_traces=wl["n_traces"],
                             openmp=True)


def test_philox_known_answers_on_device(afm):
    rows = [[int(x, 16) for x in l.split()] for l in open(KAT)
            if l.strip() and not l.startswith("#")]
    for w in rows:
        out = afm.afm_philox4x32_10([w[0:4]], w[4:6])
        assert [int(x) for x in out[0]] == w[6:10]


def test_philox_matches_oracle_on_random_counters(afm):
    rng = np.random.default_rng(5)
    ctr = rng.integers(0, 2 ** 32, size=(1000, 4), dtype=np.uint64).astype(np.uint32)
    key = [0x9E3779B9, 0x12345678]
    out = afm.afm_philox4x32_10(ctr, key)
    for i in range(0, 1000, 37):
        assert [int(x) for x in out[i]] == orc.philox4x32_10(ctr[i], key)


@pytest.mark.parametrize("cfg_i,law", [(0, None), (0, wlm.LAW_NONE), (2, None), (3, None)])
def test_trajectory_matches_oracle(afm, cfg_i, law):
    """Same RK4 states, step by step, for each force law (20 cycles)."""
    wl = wlm.scaled(wlm.config(cfg_i), n_cycles=20, n_skip_cycles=10)
    if law is not None:
        wl = dict(wl, law=law)
    M = orc.model_from(wl)
    bad, zs, vs = orc.integrate(M, wl["truth"], wl["z0"], wl["v0"])
    assert bad == 0
    gz, gv = afm.afm_trajectory(wl["truth"], afm.cfg_from(wl), wl["z0"], wl["v0"])
    A0 = wl["cantilever"]["A0"]
    w = 2 * np.pi * wl["cantilever"]["f_drive"]
    assert np.max(np.abs(gz - zs)) / A0 < 1e-11
    assert np.max(np.abs(gv - vs)) / (A0 * w) < 1e-11


def test_forward_cfg0_all_particles_ragged(afm):
    """configs[0] sizes; 100 particles = several CTAs and a ragged tail."""
    wl = wlm.config(0)
    trace = oracle_trace(wl)
    params = wlm.draw_params(wl, 100, seed=11)
    params[0] = wl["truth"]
    Jo = _oracle_forward(wl, params, trace)
    Jg = _gpu_forward(afm, wl, params, trace)
    assert np.all(np.isfinite(Jo))
    assert rel_err(Jg, Jo).max() < TOL_F64
    # J(truth) on a noisy trace ~ W sigma^2 (both sides)
    assert Jg[0] == pytest.approx(wl["n_window"] * wl["sigma"] ** 2, rel=0.2)


@pytest.mark.parametrize("block,tile", [(32, 0), (64, 0), (128, 0), (32, 50), (64, 33)])
def test_forward_launch_shapes(afm, block, tile):
    """Every CTA size and odd tile sizes (ragged last tile, window start inside a
    tile) give the same misfits."""
    wl = wlm.scaled(wlm.config(0), n_cycles=7, n_skip_cycles=3)
    trace = oracle_trace(wl)
    params = wlm.draw_params(wl, 131, seed=12)
    Jo = _oracle_forward(wl, params, trace)
    afm.afm_set_option("block", block)
    afm.afm_set_option("tile", tile)
    try:
        Jg = _gpu_forward(afm, wl, params, trace)
    finally:
        afm.afm_set_option("block", 0)
        afm.afm_set_option("tile", 0)
    assert rel_err(Jg, Jo).max() < TOL_F64


@pytest.mark.parametrize("cfg_i", [1, 2])
def test_forward_kernel_forms_agree(afm, cfg_i):
    """The throughput form (fewest FP64 instructions) and the latency form
    (vdW term folded so that one dependent FMA follows the correction) of the
    FP64 kernel: each within 1e-9 of the oracle, within rounding of one another."""
    wl = wlm.scaled(wlm.config(cfg_i), n_cycles=24, n_skip_cycles=12)
    trace = oracle_trace(wl)
    n = 517
    params = wlm.draw_params(wl, n, seed=21)
    z0v0 = wlm.draw_initial_states(wl, n, seed=22) if cfg_i == 1 else None
    Jo = _oracle_forward(wl, params, trace, z0v0)
    out = {}
    for form in (1, 2):
        afm.afm_set_option("form", form)
        try:
            out[form] = _gpu_forward(afm, wl, params, trace, z0v0)
        finally:
            afm.afm_set_option("form", 0)
        assert rel_err(out[form], Jo).max() < TOL_F64, form
    assert not np.array_equal(out[1], out[2])      # they really are two code paths
    assert rel_err(out[1], out[2]).max() < 1e-10


def test_forward_cfg1_shape_random_phases(afm):
    """configs[1] shape (S=256, random initial phases, log-uniform theta) at 40
    cycles on 2065 particles."""
    wl = wlm.scaled(wlm.config(1), n_cycles=40, n_skip_cycles=20)
    trace = oracle_trace(wl)
    n = 2065
    params = wlm.draw_params(wl, n, seed=1)
    z0v0 = wlm.draw_initial_states(wl, n, seed=2)
    Jo = _oracle_forward(wl, params, trace, z0v0)
    Jg = _gpu_forward(afm, wl, params, trace, z0v0)
    e = rel_err(Jg, Jo)
    assert e.max() < TOL_F64, (e.max(), int(e.argmax()))


def test_forward_cfg2_shape_viscoelastic(afm):
    wl = wlm.scaled(wlm.config(2), n_cycles=30, n_skip_cycles=15)
    trace = oracle_trace(wl)
    params = wlm.draw_params(wl, 515, seed=3)
    Jo = _oracle_forward(wl, params, trace)
    Jg = _gpu_forward(afm, wl, params, trace)
    assert rel_err(Jg, Jo).max() < TOL_F64


def test_forward_cfg3_shape_lj_exp(afm):
    wl = wlm.scaled(wlm.config(3), n_cycles=16, n_skip_cycles=8)
    trace = oracle_trace(wl)
    params = wlm.draw_params(wl, 300, seed=4)
    Jo = _oracle_forward(wl, params, trace)
    Jg = _gpu_forward(afm, wl, params, trace)
    fin = np.isfinite(Jo)
    assert np.array_equal(np.isfinite(Jg), fin)
    assert rel_err(Jg, Jo).max() < TOL_F64


def test_forward_cfg4_shape_many_traces(afm):
    """configs[4] shape: several traces, each with its own segment of particles
    (70 per trace: ragged CTAs inside every segment)."""
    wl = wlm.scaled(wlm.config(4), n_cycles=12, n_skip_cycles=6, n_traces=5)
    truths = wlm.pixel_truths(wl)
    trace = oracle_trace(wl, truths=truths)
    per = 70
    params = wlm.draw_params(wl, per * 5, seed=6)
    Jo = _oracle_forward(wl, params, trace)
    Jg = _gpu_forward(afm, wl, params, trace)
    assert rel_err(Jg, Jo).max() < TOL_F64
    # the segments really use different traces: swapping two traces changes J
    Jg2 = _gpu_forward(afm, wl, params, trace[::-1])
    assert np.abs(Jg2[:per] - Jg[:per]).max() > 0


def test_forward_edge_cases(afm):
    wl = wlm.scaled(wlm.config(0), n_cycles=4, n_skip_cycles=0)   # window = everything
    trace = oracle_trace(wl)
    one = np.array([wl["truth"]])
    assert rel_err(_gpu_forward(afm, wl, one, trace), _oracle_forward(wl, one, trace)).max() < TOL_F64
    # a single step in total
    w1 = wlm.scaled(wlm.config(0), steps_per_cycle=1, n_cycles=1, n_skip_cycles=0)
    tr1 = np.array([[1e-9]])
    p = wlm.draw_params(w1, 3, seed=1)
    assert rel_err(_gpu_forward(afm, w1, p, tr1), _oracle_forward(w1, p, tr1)).max() < TOL_F64
    # noise-free trace of the truth: J(truth) is (numerically) zero
    clean = oracle_trace(wl, noise=False)
    J0 = _gpu_forward(afm, wl, one, clean)[0]
    assert J0 < 1e-12 * wl["n_window"] * wl["cantilever"]["A0"] ** 2


def test_forward_divergence_gives_inf(afm):
    """A trajectory that blows up is +Inf on both sides (reading R12).  Particles
    at the edge of blowing up are ill-conditioned: they are compared only where
    the oracle's own verdict survives a 1e-13 relative change of theta
    (SURVEY.md 8(c) c-15 protocol)."""
    base = wlm.scaled(wlm.config(3), n_cycles=6, n_skip_cycles=3)
    trace = np.zeros((1, base["n_window"]))
    params = wlm.draw_params(base, 64, seed=9)
    # tip driven into the d^-8 wall: most diverge, some survive
    wl = dict(base, cantilever=dict(base["cantilever"], z_c=15e-9))
    Jo = _oracle_forward(wl, params, trace)
    Jo2 = _oracle_forward(wl, params * (1 + 1e-13), trace)
    Jg = _gpu_forward(afm, wl, params, trace)
    assert np.isinf(Jo).any() and np.isfinite(Jo).any()
    assert not np.isnan(Jg).any()
    robust = (np.isinf(Jo) == np.isinf(Jo2)) & (rel_err(Jo2, Jo) < 1e-12)
    assert robust.sum() > 32 and np.isinf(Jo[robust]).sum() > 8
    assert np.array_equal(np.isinf(Jg)[robust], np.isinf(Jo)[robust])
    assert rel_err(Jg, Jo)[robust].max() < TOL_F64


def test_forward_host_entry_matches_device_entry(afm):
    wl = wlm.scaled(wlm.config(0), n_cycles=6, n_skip_cycles=3)
    trace = oracle_trace(wl)
    params = wlm.draw_params(wl, 77, seed=13)
    Jd = _gpu_forward(afm, wl, params, trace)
    Jh = afm.afm_forward_batch_host(params, trace, afm.cfg_from(wl))
    assert np.array_equal(Jd, Jh)


def test_bad_arguments_are_rejected(afm):
    import torch
    wl = wlm.config(0)
    cfg = afm.cfg_from(wl)
    t = torch.zeros(wl["n_window"], dtype=torch.float64, device="cuda")
    p = torch.zeros((4, 2), dtype=torch.float64, device="cuda")
    for field, val in (("n_params", 3), ("steps_per_cycle", 0), ("n_skip_cycles", 20),
                       ("law", 9), ("n_traces", 3), ("Q", 0.0), ("reserved_", 1)):
        bad = afm.cfg_from(wl, **{field: val})
        with pytest.raises(afm.AfmError) as ei:
            afm.lib().afm_forward_batch  # symbol exists
            from paper_1109_0334_b200.afm import _check, _ptr
            import ctypes as C
            _check(afm.lib().afm_forward_batch(_ptr(p), 4, _ptr(t), C.byref(bad), None,
                                               _ptr(p), None))
        assert ei.value.code == afm.EINVAL, field
    assert "n_traces" in afm.afm_last_error() or afm.afm_last_error()
    J = afm.afm_forward_batch(p + 1e-19, t, cfg)   # a valid call still works afterwards
    torch.cuda.synchronize()
    assert J.shape == (4,)


@pytest.mark.parametrize("precision", [0, 1])
def test_warp_packing_changes_no_result(afm, precision):
    """afm_set_option("pack"): the particles of a DMT batch are integrated in the
    order (trace, initial phase bin, stiffness) instead of the caller's order.
    Every misfit must be bit-identical, for one trace with random phases and for
    several traces, forward and inside an inversion."""
    import torch
    wl = wlm.scaled(wlm.config(1), n_cycles=12, n_skip_cycles=6)
    trace = oracle_trace(wl)
    n = 3000 + 7
    params = wlm.draw_params(wl, n, seed=51)
    z0v0 = wlm.draw_initial_states(wl, n, seed=52)
    out = {}
    for pack in (1, 2):
        afm.afm_set_option("pack", pack)
        try:
            out[pack] = _gpu_forward(afm, wl, params, trace, z0v0, precision=precision)
            w4 = wlm.scaled(wlm.config(4), n_cycles=8, n_skip_cycles=4, n_traces=3)
            tr4 = oracle_trace(w4, truths=wlm.pixel_truths(w4))
            p4 = wlm.draw_params(w4, 3 * 211, seed=53)
            out[pack, 4] = _gpu_forward(afm, w4, p4, tr4, precision=precision)
            w2 = wlm.scaled(wlm.config(2), n_cycles=8, n_skip_cycles=4, n_particles=300,
                            n_iters=4)
            g = afm.afm_pso_invert(afm.bounds_from(w2), afm.swarm_from(w2), 0,
                                   torch.as_tensor(oracle_trace(w2), device="cuda"),
                                   afm.cfg_from(w2, precision=precision), dump=True)
            out[pack, 2] = g["dump"].cpu().numpy()
        finally:
            afm.afm_set_option("pack", 0)
    assert np.array_equal(out[1], out[2])
    assert np.array_equal(out[1, 4], out[2, 4])
    assert np.array_equal(out[1, 2], out[2, 2])
    if precision == 0:
        Jo = _oracle_forward(wl, params, trace, z0v0)
        assert rel_err(out[2], Jo).max() < TOL_F64


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("cfg_i,segs,workers,boost", [
    (1, 0, 0, 0), (1, 5, 1, 0), (2, 3, 8, 0), (3, 7, 2, 0), (4, 1, 4, 0), (4, 2047, 3, 0),
    (1, 24, 1, 64), (1, 48, 2, 1), (1, 16, 1, 2)])
def test_segment_queue_changes_no_result(afm, cfg_i, segs, workers, boost, precision):
    """afm_set_option("queue"): the time loop of every warp of particles is cut into
    segments that persistent workers take from a priority queue in global memory
    keyed by the segment index (integrate_misfit_f64_q, integrate_misfit_f32_q).
    Misfits, and the swarm of an inversion, must be bit-identical to the
    one-CTA-per-warp kernel: ragged particle counts, several traces, every segment
    count from one to one tile per segment, fewer workers than chains (chains wait,
    the lowest segment first), the boost of the chains that are behind on, off and
    at its most eager (a worker pauses whenever 1/64 of the chains are a segment
    ahead), all law families; and they must match the oracle."""
    import torch
    over = dict(n_cycles=12, n_skip_cycles=6)
    if cfg_i == 4:
        over["n_traces"] = 3
    wl = wlm.scaled(wlm.config(cfg_i), **over)
    T = wl["n_traces"]
    truths = None if wl["truth"] is not None else wlm.pixel_truths(wl)
    trace = oracle_trace(wl, truths=truths)
    # (1, 5, 1): 626 chains on 592 workers, so chains also wait for a free worker;
    # the boost cases: 1 251 chains on 592 or 1 184 workers
    n = 40013 if boost else 20013 if (cfg_i, workers) == (1, 1) else T * (300 + 13)
    params = wlm.draw_params(wl, n, seed=61)
    z0v0 = wlm.draw_initial_states(wl, n, seed=62) if cfg_i == 1 else None
    wp = wlm.scaled(wl, n_particles=77, n_iters=4)
    out = {}
    for queue in (1, 2):
        afm.afm_set_option("queue", queue)
        afm.afm_set_option("segs", segs)
        afm.afm_set_option("workers", workers)
        afm.afm_set_option("boost", boost)
        afm.afm_set_option("form", 1)           # the queue serves the throughput form
        try:
            out[queue] = _gpu_forward(afm, wl, params, trace, z0v0, precision=precision)
            afm.afm_queue_status()              # no worker gave up (raises otherwise)
            g = afm.afm_pso_invert(afm.bounds_from(wp), afm.swarm_from(wp), 3,
                                   torch.as_tensor(trace, device="cuda"),
                                   afm.cfg_from(wp, precision=precision), dump=True)
            out[queue, "pso"] = g["dump"].cpu().numpy()
        finally:
            for name in ("queue", "segs", "workers", "boost", "form"):
                afm.afm_set_option(name, 0)
    assert np.array_equal(out[1], out[2])
    assert np.array_equal(out[1, "pso"], out[2, "pso"])
    if precision == 0:
        pick = np.arange(0, n, 16) if boost else np.arange(n)   # the oracle on every 16th
        Jo = _oracle_forward(wl, params[pick], trace, None if z0v0 is None else z0v0[pick])
        assert rel_err(out[2][pick], Jo).max() < TOL_F64


@pytest.mark.parametrize("lanes", [1, 2, 8, 32])
def test_latency_form_lanes_per_warp(afm, lanes):
    """Latency form with 1..32 particles per warp (the other lanes shadow them):
    bit-identical misfits and swarm, ragged counts included."""
    import torch
    wl = wlm.scaled(wlm.config(2), n_cycles=10, n_skip_cycles=5, n_particles=77, n_iters=4)
    trace = oracle_trace(wl)
    params = wlm.draw_params(wl, 77, seed=61)
    out = {}
    for l in (32, lanes):
        afm.afm_set_option("lanes", l)
        afm.afm_set_option("form", 2)
        try:
            J = _gpu_forward(afm, wl, params, trace)
            g = afm.afm_pso_invert(afm.bounds_from(wl), afm.swarm_from(wl), 0,
                                   torch.as_tensor(trace, device="cuda"), afm.cfg_from(wl),
                                   dump=True)
            out[l] = (J, g["dump"].cpu().numpy(), g["theta_star"])
        finally:
            afm.afm_set_option("lanes", 0)
            afm.afm_set_option("form", 0)
    assert np.array_equal(out[32][0], out[lanes][0])
    assert np.array_equal(out[32][1], out[lanes][1])
    assert np.array_equal(out[32][2], out[lanes][2])
    assert rel_err(out[lanes][0], _oracle_forward(wl, params, trace)).max() < TOL_F64


@pytest.mark.parametrize("precision", [0, 1])
def test_segment_queue_random_schedules_never_change_a_result(afm, precision):
    """The priority queue under random schedules: segment counts, workers per
    sub-partition (more and fewer than chains) and boost thresholds drawn at random,
    batches of 1 251 and 2 188 chains on configs[1]'s shape (random phases, so the
    chains are very unequal and the boost fires).  Every run must reproduce the
    one-CTA-per-warp kernel bit for bit: a missing fence or a lost slot in the queue
    would show here as a wrong or stale misfit.  AFM_QUEUE_STRESS=n repeats the
    draw n times per batch instead of 10 (profiles/r2_bounds_check.md)."""
    import os
    import torch
    reps = int(os.environ.get("AFM_QUEUE_STRESS", "10"))
    wl = wlm.scaled(wlm.config(1), n_cycles=40, n_skip_cycles=20)
    trace = oracle_trace(wl)
    rng = np.random.default_rng(5 + precision)
    for n in (40013, 70001):
        params = wlm.draw_params(wl, n, seed=71)
        z0v0 = wlm.draw_initial_states(wl, n, seed=72)
        afm.afm_set_option("queue", 1)
        afm.afm_set_option("form", 1)           # the queue serves the throughput form
        try:
            ref = _gpu_forward(afm, wl, params, trace, z0v0, precision=precision)
            afm.afm_set_option("queue", 2)
            for _ in range(reps):
                afm.afm_set_option("segs", int(rng.integers(0, 160)))
                afm.afm_set_option("workers", int(rng.choice([0, 1, 2, 3, 4, 6])))
                afm.afm_set_option("boost", int(rng.choice([0, 1, 2, 5, 64])))
                afm.afm_set_option("boost2", int(rng.choice([0, 1])))
                got = _gpu_forward(afm, wl, params, trace, z0v0, precision=precision)
                assert np.array_equal(got, ref)
        finally:
            for name in ("queue", "form", "segs", "workers", "boost", "boost2"):
                afm.afm_set_option(name, 0)

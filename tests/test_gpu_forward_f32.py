"""GPU parity of the FP32 integrate-and-misfit kernel (cfg.precision = AFM_F32)
against the FP64 CPU oracle on the same seeded inputs.

Tolerance (BASELINE.json:north_star): per-particle misfit within 1e-3 relative.
The FP32 kernel integrates in kernel units with a two-float compensated state
(R14); a resonant cantilever (Q = 100..400) amplifies every rounding
of the linear terms by ~Q, so the error has a tail: the bulk sits at 1e-7..1e-4.
Every particle must meet 1e-3 unless the oracle itself is ill-conditioned
there (SURVEY.md c-15 protocol, _check_bulk_and_outliers).
"""
import numpy as np
import pytest

from oracle import binding as orc
from paper_1109_0334_b200 import workloads as wlm
from parity_helpers import oracle_trace, record_parity, rel_err

pytestmark = pytest.mark.gpu

TOL_F32 = 1e-3


@pytest.fixture(scope="module")
def afm():
    import torch
    assert torch.cuda.is_available()
    from paper_1109_0334_b200 import afm as m
    m.lib()
    yield m
    for k in ("block", "tile", "ppt"):
        m.afm_set_option(k, 0)


def _gpu(afm, wl, params, trace, z0v0=None, precision=None):
    import torch
    cfg = afm.cfg_from(wl, precision=afm.F32 if precision is None else precision)
    p = torch.as_tensor(np.ascontiguousarray(params), device="cuda")
    t = torch.as_tensor(np.ascontiguousarray(trace), device="cuda")
    zv = None if z0v0 is None else torch.as_tensor(np.ascontiguousarray(z0v0), device="cuda")
    J = afm.afm_forward_batch(p, t, cfg, z0v0=zv)
    torch.cuda.synchronize()
    return J.cpu().numpy()


def _oracle(wl, params, trace, z0v0=None):
    return orc.forward_batch(orc.model_from(wl), params, trace, z0v0=z0v0,
                             z0=wl["z0"], v0=wl["v0"], n_traces=wl["n_traces"],
                             openmp=True)


def _check_bulk_and_outliers(wl, params, trace, z0v0, Jg, Jo, label, max_outliers):
    """SURVEY.md 8(c) c-15 protocol.  Every particle must meet TOL_F32 unless the
    ORACLE ITSELF is ill-conditioned there: a 1e-10 relative change of theta or
    of the initial state moves the oracle's own J by more than ILL = 2.1e-7
    relative, i.e. the amplification exceeds 2.1e3 and a ONE-ulp FP32
    perturbation (2^-23) of the inputs alone already moves J by TOL_F32/4 (the
    paper cites chaotic tip dynamics, PAPER.md ref [12]).  At most
    `max_outliers` such particles, each one verified."""
    ILL = 0.25 * TOL_F32 / 2.0 ** -23 * 1e-10
    fin = np.isfinite(Jo)
    assert np.array_equal(np.isfinite(Jg), fin)
    e = rel_err(Jg, Jo)
    print("%s f32: median %.2e p99 %.2e p99.9 %.2e max %.2e" %
          (label, np.median(e), np.percentile(e, 99), np.percentile(e, 99.9), e.max()))
    out = np.flatnonzero(e >= TOL_F32)
    assert out.size <= max_outliers, (out.size, e[out])
    M = orc.model_from(wl)
    moves = []
    for i in out:
        p = params[i:i + 1]
        z = None if z0v0 is None else z0v0[i:i + 1]
        kw = dict(z0=wl["z0"], v0=wl["v0"])
        J0 = orc.forward_batch(M, p, trace, z0v0=z, **kw)[0]
        moved = 0.0
        for eps in (1e-10, -1e-10):
            J1 = orc.forward_batch(M, p * (1 + eps), trace, z0v0=z, **kw)[0]
            moved = max(moved, abs(J1 - J0) / J0)
            if z is not None:
                J2 = orc.forward_batch(M, p, trace, z0v0=z * (1 + eps), **kw)[0]
            else:
                J2 = orc.forward_batch(M, p, trace, z0=wl["z0"] + eps * 1e-9,
                                       v0=wl["v0"] * (1 + eps))[0]
            moved = max(moved, abs(J2 - J0) / J0)
        print("  outlier %d: err %.2e, oracle moves %.2e under a 1e-10 perturbation"
              % (i, e[i], moved))
        moves.append(moved)
    # recorded before asserting: excused by the repository's rule (ILL, TOL/4 at one
    # FP32 ulp) and by SURVEY.md c-15 as written (the full TOL at one ulp = 4 ILL)
    record_parity("%s shape, %d particles" % (label, e.size), "f32", e, TOL_F32, out.size,
                  sum(m > ILL for m in moves), sum(m > 4 * ILL for m in moves))
    for i, moved in zip(out, moves):
        assert moved > ILL, (int(i), e[i], moved)
    return e


def test_f32_cfg0_ragged(afm):
    wl = wlm.config(0)
    trace = oracle_trace(wl)
    params = wlm.draw_params(wl, 100, seed=11)
    params[0] = wl["truth"]
    Jo = _oracle(wl, params, trace)
    Jg = _gpu(afm, wl, params, trace)
    e = rel_err(Jg, Jo)
    assert e.max() < TOL_F32, (e.max(), int(e.argmax()))
    # it really is another kernel: not bit-identical to the FP64 path
    J64 = _gpu(afm, wl, params, trace, precision=afm.F64)
    assert not np.array_equal(J64, Jg)


@pytest.mark.parametrize("block,tile,ppt", [(32, 0, 1), (64, 0, 1), (128, 0, 2),
                                            (32, 50, 2), (64, 33, 1)])
def test_f32_launch_shapes(afm, block, tile, ppt):
    """CTA sizes, odd tile sizes (ragged last tile, window start inside a tile)
    and two particles per thread: all within tolerance of the oracle, and a
    lane's arithmetic does not depend on the shape (bit-equal among shapes)."""
    wl = wlm.scaled(wlm.config(0), n_cycles=7, n_skip_cycles=3)
    trace = oracle_trace(wl)
    params = wlm.draw_params(wl, 131, seed=12)
    Jo = _oracle(wl, params, trace)
    Jref = _gpu(afm, wl, params, trace)
    afm.afm_set_option("block", block)
    afm.afm_set_option("tile", tile)
    afm.afm_set_option("ppt", ppt)
    try:
        Jg = _gpu(afm, wl, params, trace)
    finally:
        for k in ("block", "tile", "ppt"):
            afm.afm_set_option(k, 0)
    assert rel_err(Jg, Jo).max() < TOL_F32
    if tile == 0:
        # the per-tile fold of the misfit sum depends on the tile size only
        assert np.array_equal(Jg, Jref)


def test_f32_cfg1_full_length_random_phases(afm):
    """configs[1] at its full 200 cycles x 256 steps on 4099 particles (ragged)."""
    wl = wlm.config(1)
    trace = oracle_trace(wl)
    n = 4099
    params = wlm.draw_params(wl, n, seed=1)
    z0v0 = wlm.draw_initial_states(wl, n, seed=2)
    Jo = _oracle(wl, params, trace, z0v0)
    Jg = _gpu(afm, wl, params, trace, z0v0)
    e = _check_bulk_and_outliers(wl, params, trace, z0v0, Jg, Jo, "cfg1", 8)
    assert np.percentile(e, 99) < 1e-4


def test_f32_cfg2_shape_viscoelastic(afm):
    wl = wlm.scaled(wlm.config(2), n_cycles=60, n_skip_cycles=30)
    trace = oracle_trace(wl)
    params = wlm.draw_params(wl, 1031, seed=3)
    Jo = _oracle(wl, params, trace)
    Jg = _gpu(afm, wl, params, trace)
    _check_bulk_and_outliers(wl, params, trace, None, Jg, Jo, "cfg2", 2)


def test_f32_cfg3_full_length_lj_exp(afm):
    """configs[3] at its full 150 cycles x 512 steps, Q = 400: the stiff case.
    SURVEY.md c-14/c-15: a tail of ill-conditioned particles remains in FP32;
    every particle above 1e-3 must be one the oracle itself cannot resolve."""
    wl = wlm.config(3)
    trace = oracle_trace(wl)
    params = wlm.draw_params(wl, 1024, seed=4)
    Jo = _oracle(wl, params, trace)
    Jg = _gpu(afm, wl, params, trace)
    e = _check_bulk_and_outliers(wl, params, trace, None, Jg, Jo, "cfg3", 10)
    assert np.percentile(e, 99) < TOL_F32


def test_f32_cfg4_shape_many_traces(afm):
    wl = wlm.scaled(wlm.config(4), n_cycles=12, n_skip_cycles=6, n_traces=5)
    truths = wlm.pixel_truths(wl)
    trace = oracle_trace(wl, truths=truths)
    per = 70
    params = wlm.draw_params(wl, per * 5, seed=6)
    Jo = _oracle(wl, params, trace)
    Jg = _gpu(afm, wl, params, trace)
    assert rel_err(Jg, Jo).max() < TOL_F32


def test_f32_edge_cases(afm):
    wl = wlm.scaled(wlm.config(0), n_cycles=4, n_skip_cycles=0)
    trace = oracle_trace(wl)
    one = np.array([wl["truth"]])
    assert rel_err(_gpu(afm, wl, one, trace), _oracle(wl, one, trace)).max() < TOL_F32
    w1 = wlm.scaled(wlm.config(0), steps_per_cycle=1, n_cycles=1, n_skip_cycles=0)
    tr1 = np.array([[1e-9]])
    p = wlm.draw_params(w1, 3, seed=1)
    assert rel_err(_gpu(afm, w1, p, tr1), _oracle(w1, p, tr1)).max() < TOL_F32
    # linear oscillator (law NONE) on a noise-free trace of itself: J ~ rounding
    wn = dict(wlm.scaled(wlm.config(0), n_cycles=8, n_skip_cycles=4), law=wlm.LAW_NONE)
    clean = oracle_trace(wn, noise=False)
    J0 = _gpu(afm, wn, one, clean)[0]
    A0 = wn["cantilever"]["A0"]
    assert J0 < 1e-10 * wn["n_window"] * A0 ** 2


def test_f32_divergence_gives_inf(afm):
    """Blow-ups are +Inf (R12).  Whether RK4 blows up at the d^-8 wall is itself
    chaotic for the marginal particles, so verdicts are compared where the
    oracle's own verdict survives 1e-6..1e-4 relative changes of theta and z0."""
    base = wlm.scaled(wlm.config(3), n_cycles=6, n_skip_cycles=3)
    trace = np.zeros((1, base["n_window"]))
    params = wlm.draw_params(base, 64, seed=9)
    wl = dict(base, cantilever=dict(base["cantilever"], z_c=15e-9))
    Jo = _oracle(wl, params, trace)
    Jg = _gpu(afm, wl, params, trace)
    assert not np.isnan(Jg).any()
    robust = np.ones(len(Jo), dtype=bool)
    M = orc.model_from(wl)
    for eps in (1e-6, -1e-6, 1e-5, -1e-5, 1e-4, -1e-4):
        J1 = _oracle(wl, params * (1 + eps), trace)
        J2 = orc.forward_batch(M, params, trace, z0=wl["z0"] + eps * 1e-9, v0=wl["v0"],
                               openmp=True)
        robust &= (np.isinf(J1) == np.isinf(Jo)) & (np.isinf(J2) == np.isinf(Jo))
    assert robust.sum() > 16 and np.isinf(Jo[robust]).sum() > 4
    assert np.array_equal(np.isinf(Jg)[robust], np.isinf(Jo)[robust])


def test_f32_pso_teacher_forced(afm):
    """DESIGN.md R17 / SURVEY.md c-17: FP32 misfits differ from FP64 by up to 1e-3, so
    the swarm may legitimately take another path than the FP64 oracle's.  Teacher
    forcing, both halves: (1) at every iteration the GPU's own positions x are
    evaluated by the oracle (J within 1e-3); (2) the ORACLE's PSO loop is replayed
    with the GPU's own J as its cost (a scripted callback: the k-th evaluation
    returns the J the GPU recorded for it), and every x, v, pbest and pbestJ of the
    GPU run must equal that replay bit for bit, as must theta* and J*."""
    import torch
    wl = wlm.scaled(wlm.config(2), n_cycles=20, n_skip_cycles=10, n_particles=96,
                    n_iters=6)
    trace = oracle_trace(wl)
    t = torch.as_tensor(trace, device="cuda")
    cfg = afm.cfg_from(wl, precision=afm.F32)
    seed = 5
    g = afm.afm_pso_invert(afm.bounds_from(wl), afm.swarm_from(wl), seed, t, cfg,
                           dump=True, hist=True)
    d = g["dump"].cpu().numpy()            # [it][P][3D+2]
    D, P = wl["n_params"], d.shape[1]
    M = orc.model_from(wl)
    for it in range(d.shape[0]):
        th = wlm.theta_of_coords(wl, d[it, :, 0:D])
        Jo = orc.forward_batch(M, th, trace, z0=wl["z0"], v0=wl["v0"], openmp=True)
        assert rel_err(d[it, :, 3 * D], Jo).max() < TOL_F32, it
    # (2) Eq. 8 on the CPU from the GPU's own J
    calls = {"k": 0, "theta": []}

    def gpu_cost(theta, _U):
        k = calls["k"]
        calls["k"] += 1
        calls["theta"].append(theta)
        return d[k // P, k % P, 3 * D]

    o = orc.pso_core(gpu_cost, D, orc.box_from(wl), orc.swarm_from(wl), seed, trace)
    assert calls["k"] == d.shape[0] * P
    assert np.array_equal(o["dump"], d)                 # x, v, pbest, J, pbestJ
    assert np.array_equal(o["gbest_hist"], g["gbest_hist"].cpu().numpy())
    assert np.array_equal(o["J_star"], g["J_star"])
    # theta* = 10^x through two different pow() implementations: last-bit agreement
    assert rel_err(g["theta_star"], o["theta_star"]).max() < 1e-15
    # the oracle asked for the cost at exactly the parameters the GPU integrated
    th_all = wlm.theta_of_coords(wl, d[:, :, 0:D].reshape(-1, D))
    assert rel_err(np.array(calls["theta"]), th_all).max() < 1e-15

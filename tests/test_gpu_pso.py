"""GPU parity: afm_pso_invert / afm_pso_init / afm_pso_step (through the C ABI)
against the CPU oracle's PSO on the same seeds.

BASELINE.json:north_star: "PSO runs replay identical Philox streams, the
per-iteration swarm state in FP64 must agree to 1e-9 relative, and the final
theta* must agree with the oracle's ... within 1e-3 relative".  The PSO
arithmetic itself is written without FMA contraction on both sides, so x, v and
pbest normally agree bit for bit; J and pbestJ carry the forward solve's
rounding differences (~1e-11).
"""
import numpy as np
import pytest

from oracle import binding as orc
from paper_1109_0334_b200 import workloads as wlm
from parity_helpers import oracle_trace, rel_err

pytestmark = pytest.mark.gpu

TOL = 1e-9


@pytest.fixture(scope="module")
def afm():
    import torch
    assert torch.cuda.is_available()
    from paper_1109_0334_b200 import afm as m
    m.lib()
    return m


def _both(afm, wl, trace, seed=None, dump=True, j_target=0.0, async_chunk=0):
    import torch
    seed = wl["pso_seed"] if seed is None else seed
    cfg = afm.cfg_from(wl)
    g = afm.afm_pso_invert(afm.bounds_from(wl),
                           afm.swarm_from(wl, j_target=j_target, async_chunk=async_chunk),
                           seed, torch.as_tensor(np.ascontiguousarray(trace), device="cuda"),
                           cfg, dump=dump, hist=True)
    o = orc.pso_invert(orc.model_from(wl), orc.box_from(wl),
                       orc.swarm_from(wl, j_target=j_target, async_chunk=async_chunk), seed,
                       trace, wl["z0"], wl["v0"], n_traces=wl["n_traces"], dump=dump,
                       openmp=True)
    return g, o


def _compare_runs(g, o, D):
    gd = g["dump"].cpu().numpy()
    od = o["dump"]
    assert gd.shape == od.shape
    # x, v, pbest: scale-aware relative error (coordinates are O(1..1000))
    for name, sl in (("x", slice(0, D)), ("v", slice(D, 2 * D)), ("pbest", slice(2 * D, 3 * D))):
        a, b = gd[..., sl], od[..., sl]
        scale = np.maximum(np.abs(b), 1.0) if name != "v" else np.maximum(np.abs(b), 1e-3)
        err = np.abs(a - b) / scale
        assert err.max() < TOL, (name, err.max(), np.unravel_index(err.argmax(), err.shape))
    for name, col in (("J", 3 * D), ("pbestJ", 3 * D + 1)):
        e = rel_err(gd[..., col], od[..., col])
        assert e.max() < TOL, (name, e.max())
    gh = g["gbest_hist"].cpu().numpy()
    assert rel_err(gh[..., D], o["gbest_hist"][..., D]).max() < TOL
    assert np.abs(gh[..., :D] - o["gbest_hist"][..., :D]).max() < 1e-9 * 1000
    assert rel_err(g["theta_star"], o["theta_star"]).max() < 1e-9
    assert rel_err(g["J_star"], o["J_star"]).max() < TOL


def test_pso_init_is_bit_exact(afm):
    """x0, v0 of the GPU swarm == the oracle's iteration-0 dump, bit for bit."""
    wl = wlm.scaled(wlm.config(2), n_cycles=2, n_skip_cycles=1, n_particles=333, n_iters=1)
    trace = oracle_trace(wl)
    o = orc.pso_invert(orc.model_from(wl), orc.box_from(wl), orc.swarm_from(wl), 12345,
                       trace, wl["z0"], wl["v0"], dump=True)
    st = afm.afm_pso_init(afm.bounds_from(wl), afm.swarm_from(wl), 3, 1, 12345)
    assert np.array_equal(st["x"].cpu().numpy(), o["dump"][0, :, 0:3])
    assert np.array_equal(st["v"].cpu().numpy(), o["dump"][0, :, 3:6])
    assert np.array_equal(st["pbest"].cpu().numpy(), o["dump"][0, :, 0:3])
    assert np.all(np.isinf(st["pbestJ"].cpu().numpy()))
    lo, hi = np.array(wl["bounds"]["lo"]), np.array(wl["bounds"]["hi"])
    x = st["x"].cpu().numpy()
    assert np.all(x >= lo) and np.all(x <= hi)


def test_cfg0_full_inversion_replays_the_oracle(afm):
    """configs[0] exactly as BASELINE.json states it: 64 particles, 20 iterations."""
    wl = wlm.config(0)
    trace = oracle_trace(wl)
    g, o = _both(afm, wl, trace)
    _compare_runs(g, o, 2)
    assert g["n_iters_done"] == 20
    # invariants on the GPU run itself
    d = g["dump"].cpu().numpy()
    assert np.all(d[1:, :, 7] <= d[:-1, :, 7])                # pbestJ never increases
    gh = g["gbest_hist"].cpu().numpy()
    assert np.all(gh[1:, 0, 2] <= gh[:-1, 0, 2])
    assert np.allclose(gh[:, 0, 2], d[..., 7].min(axis=1), rtol=0, atol=0)
    # J* <= J(truth) cannot be required of 20 iterations; it is near W sigma^2
    assert g["J_star"][0] < 3 * wl["n_window"] * wl["sigma"] ** 2


def test_cfg2_shape_inversion(afm):
    """DMT + viscoelastic, 3 unknowns with one linear coordinate; 200 particles
    (ragged CTAs), 12 iterations, 16 cycles."""
    wl = wlm.scaled(wlm.config(2), n_cycles=16, n_skip_cycles=8, n_particles=200, n_iters=12)
    trace = oracle_trace(wl)
    g, o = _both(afm, wl, trace, seed=7)
    _compare_runs(g, o, 3)


def test_cfg3_shape_inversion(afm):
    wl = wlm.scaled(wlm.config(3), n_cycles=8, n_skip_cycles=4, n_particles=96, n_iters=10)
    trace = oracle_trace(wl)
    g, o = _both(afm, wl, trace, seed=3)
    _compare_runs(g, o, 4)


def test_cfg4_shape_independent_swarms_per_trace(afm):
    """Several pixels, each with its own trace, swarm and global best."""
    wl = wlm.scaled(wlm.config(4), n_cycles=10, n_skip_cycles=5, n_traces=4,
                    n_particles=80, n_iters=8)
    truths = wlm.pixel_truths(wl)
    trace = oracle_trace(wl, truths=truths)
    g, o = _both(afm, wl, trace, seed=0)
    _compare_runs(g, o, 3)
    # a pixel's result does not depend on its neighbours: rerun pixel 2 alone
    # (its particles keep their global indices only if it is first, so compare J*
    # ordering instead of values)
    assert len(set(np.round(g["J_star"] / g["J_star"].min(), 6))) > 1


def test_noise_free_truth_recovery(afm):
    """north_star: recovery of known ground truth from a noise-free synthetic
    trace on a tiny swarm, theta* within 1e-3 relative."""
    import torch
    wl = wlm.scaled(wlm.config(0), n_iters=100)
    trace = oracle_trace(wl, noise=False)
    g = afm.afm_pso_invert(afm.bounds_from(wl), afm.swarm_from(wl), 0,
                           torch.as_tensor(trace, device="cuda"), afm.cfg_from(wl))
    assert rel_err(g["theta_star"][0], wl["truth"]).max() < 1e-3
    assert g["J_star"][0] < 1e-6 * wl["n_window"] * wl["sigma"] ** 2


def _cut_target(hist, after):
    """A cutoff strictly between two successive, distinct values of a best-cost
    history (geometric mean), first crossed at batch k >= after: the ~1e-11 relative
    difference between the two forward solvers cannot move the crossing."""
    for k in range(max(after, 1), len(hist)):
        if hist[k] < hist[k - 1] * (1 - 1e-6):
            return float(np.sqrt(hist[k] * hist[k - 1])), k
    raise AssertionError("no strict improvement after batch %d" % after)


def _both_cut(afm, wl, trace, seed, j_target):
    import torch
    g = afm.afm_pso_invert(afm.bounds_from(wl), afm.swarm_from(wl, j_target=j_target), seed,
                           torch.as_tensor(np.ascontiguousarray(trace), device="cuda"),
                           afm.cfg_from(wl), dump=True, hist=True)
    o = orc.pso_invert(orc.model_from(wl), orc.box_from(wl),
                       orc.swarm_from(wl, j_target=j_target), seed, trace, wl["z0"],
                       wl["v0"], n_traces=wl["n_traces"], dump=True, openmp=True)
    return g, o


def _compare_cut_runs(g, o, D):
    """Batches run, theta*, J* and every recorded row up to the stop."""
    n = o["n_iters_done"]
    assert g["n_iters_done"] == n
    gc = dict(g, dump=g["dump"][:n], gbest_hist=g["gbest_hist"][:n])
    oc = dict(o, dump=o["dump"][:n], gbest_hist=o["gbest_hist"][:n])
    _compare_runs(gc, oc, D)
    assert np.all(np.isnan(o["dump"][n:]))              # the oracle ran no further batch


def test_j_target_single_trace_against_the_oracle(afm):
    """Cost cutoff (R24): the target is taken from
    the ORACLE's own uncut history; both sides must stop after the same batch with
    the same swarm, and no move follows the stopping batch (the dump row of that
    batch holds the positions evaluated in it; the caller's later rows are left
    untouched)."""
    import torch
    wl = wlm.scaled(wlm.config(0), n_iters=60)
    trace = oracle_trace(wl)
    full = orc.pso_invert(orc.model_from(wl), orc.box_from(wl), orc.swarm_from(wl), 0, trace,
                          wl["z0"], wl["v0"], openmp=True)
    target, k = _cut_target(full["gbest_hist"][:, 0, 2], 20)
    g, o = _both_cut(afm, wl, trace, 0, target)
    assert o["n_iters_done"] == k + 1 < 60
    _compare_cut_runs(g, o, 2)
    assert g["J_star"][0] <= target < full["gbest_hist"][k - 1, 0, 2]
    # a target nobody reaches runs every batch; a target met by the very first batch
    # stops after one
    g, o = _both_cut(afm, wl, trace, 0, 1e-30)
    assert g["n_iters_done"] == o["n_iters_done"] == 60
    g, o = _both_cut(afm, wl, trace, 0, 1.0)
    assert g["n_iters_done"] == o["n_iters_done"] == 1
    _compare_cut_runs(g, o, 2)
    # rows after the stop are not written
    sentinel = torch.full((60, 64, 8), -7.0, dtype=torch.float64, device="cuda")
    th = afm.afm_pso_invert(afm.bounds_from(wl), afm.swarm_from(wl, j_target=1.0), 0,
                            torch.as_tensor(trace, device="cuda"), afm.cfg_from(wl),
                            dump=sentinel)
    assert th["n_iters_done"] == 1
    assert bool((sentinel[1:] == -7.0).all()) and not bool((sentinel[0] == -7.0).any())


def test_j_target_waits_for_every_trace(afm):
    """Three pixels with their own traces and swarms cross the same cutoff at
    different batches; the run ends after the LAST of them has crossed (every
    trace's best <= target), the early pixels keep improving meanwhile."""
    wl = wlm.scaled(wlm.config(4), n_cycles=10, n_skip_cycles=5, n_traces=3,
                    n_particles=48, n_iters=40)
    trace = oracle_trace(wl, truths=wlm.pixel_truths(wl))
    full = orc.pso_invert(orc.model_from(wl), orc.box_from(wl), orc.swarm_from(wl), 5, trace,
                          wl["z0"], wl["v0"], n_traces=3, openmp=True)
    h = full["gbest_hist"][:, :, 3]                      # [batch][trace]
    # cutoff from the trace that is slowest to get there, between two of its values
    slow = int(np.argmax(h[20]))
    target, _ = _cut_target(h[:, slow], 12)
    cross = [int(np.argmax(h[:, s] <= target)) for s in range(3)]
    assert all(h[c, s] <= target for s, c in enumerate(cross))
    assert len(set(cross)) > 1, cross                    # the pixels do differ
    for s in range(3):                                   # no crossing is a near tie
        assert np.min(np.abs(h[:, s] / target - 1.0)) > 1e-6
    g, o = _both_cut(afm, wl, trace, 5, target)
    assert o["n_iters_done"] == max(cross) + 1 < 40
    _compare_cut_runs(g, o, 3)
    first = int(np.argmin(cross))
    assert o["J_star"][first] <= h[cross[first], first]


def test_pso_step_on_supplied_misfits(afm):
    """afm_pso_init + afm_pso_step with J supplied by the caller: replay of the
    oracle's recorded run (teacher forcing with the ORACLE's J), bit for bit."""
    import torch
    wl = wlm.scaled(wlm.config(2), n_cycles=6, n_skip_cycles=3, n_particles=150, n_iters=6)
    trace = oracle_trace(wl)
    seed = 99
    o = orc.pso_invert(orc.model_from(wl), orc.box_from(wl), orc.swarm_from(wl), seed,
                       trace, wl["z0"], wl["v0"], dump=True)
    B, S = afm.bounds_from(wl), afm.swarm_from(wl)
    st = afm.afm_pso_init(B, S, 3, 1, seed)
    for it in range(6):
        assert np.array_equal(st["x"].cpu().numpy(), o["dump"][it, :, 0:3]), it
        assert np.array_equal(st["v"].cpu().numpy(), o["dump"][it, :, 3:6]), it
        J = torch.as_tensor(o["dump"][it, :, 9].copy(), device="cuda")
        afm.afm_pso_step(B, S, 3, 1, seed, it, it < 5, J, st)
        torch.cuda.synchronize()
        assert np.array_equal(st["pbest"].cpu().numpy(), o["dump"][it, :, 6:9]), it
        assert np.array_equal(st["pbestJ"].cpu().numpy(), o["dump"][it, :, 10]), it
        assert np.array_equal(st["gbest"].cpu().numpy()[0], o["gbest_hist"][it, 0, :3]), it
        assert st["gbestJ"].cpu().numpy()[0] == o["gbest_hist"][it, 0, 3]


@pytest.mark.parametrize("per,T", [(1, 9), (33, 7), (1, 1)])
def test_degenerate_swarm_shapes(afm, per, T):
    """One particle per swarm, ragged swarms over several traces, a single particle
    in total: the swarm still replays the oracle."""
    wl = wlm.scaled(wlm.config(4), n_cycles=6, n_skip_cycles=3, n_traces=T, n_particles=per,
                    n_iters=4)
    trace = oracle_trace(wl, truths=wlm.pixel_truths(wl))
    g, o = _both(afm, wl, trace)
    _compare_runs(g, o, wl["n_params"])


@pytest.mark.parametrize("cfg_i,T", [(2, 1), (4, 3)])
def test_ring_topology_replays_the_oracle(afm, cfg_i, T):
    """topology = 1 (ring of three, R23): same dump as the oracle's ring swarm, and
    a different swarm from the global-best one."""
    over = dict(n_cycles=8, n_skip_cycles=4, n_particles=45, n_iters=6)
    if cfg_i == 4:
        over["n_traces"] = T
    wl = wlm.scaled(wlm.config(cfg_i), **over)
    wl["swarm"]["topology"] = 1
    truths = None if wl["truth"] is not None else wlm.pixel_truths(wl)
    trace = oracle_trace(wl, truths=truths)
    g, o = _both(afm, wl, trace)
    _compare_runs(g, o, wl["n_params"])
    wl0 = wlm.scaled(wl)
    wl0["swarm"]["topology"] = 0
    g0, _ = _both(afm, wl0, trace)
    assert not np.array_equal(g0["dump"].cpu().numpy()[3], g["dump"].cpu().numpy()[3])


@pytest.mark.parametrize("cfg_i,T,per,chunk,topology",
                         [(2, 1, 45, 16, 0), (4, 3, 40, 7, 0), (2, 1, 45, 1, 0),
                          (4, 2, 33, 16, 1), (0, 1, 64, 32, 1)])
def test_async_swarm_replays_the_oracle(afm, cfg_i, T, per, chunk, topology):
    """async_chunk (R25): the swarm is processed in chunks of `chunk`
    particles that move as soon as they are evaluated.  Same dump as the oracle's
    chunked swarm -- ragged last chunk, several traces, one particle per chunk, the
    ring of three reading neighbours' bests as they stand when the chunk moves -- and
    a different swarm from the synchronous one."""
    over = dict(n_cycles=8, n_skip_cycles=4, n_particles=per, n_iters=6)
    if cfg_i == 4:
        over["n_traces"] = T
    wl = wlm.scaled(wlm.config(cfg_i), **over)
    wl["swarm"]["topology"] = topology
    truths = None if wl["truth"] is not None else wlm.pixel_truths(wl)
    trace = oracle_trace(wl, truths=truths)
    g, o = _both(afm, wl, trace, async_chunk=chunk)
    _compare_runs(g, o, wl["n_params"])
    assert g["n_iters_done"] == o["n_iters_done"] == 6
    gs, _ = _both(afm, wl, trace)
    if topology == 0:    # (in the ring only the particles at a chunk edge can tell)
        assert not np.array_equal(gs["dump"].cpu().numpy()[2], g["dump"].cpu().numpy()[2])
    # a chunk that covers the swarm is the synchronous swarm, bit for bit
    gw, _ = _both(afm, wl, trace, async_chunk=per)
    assert np.array_equal(gw["dump"].cpu().numpy(), gs["dump"].cpu().numpy())


def test_async_swarm_with_cost_cutoff_and_fp32_kernel(afm):
    """The cutoff is tested once per batch, after the last chunk (R24 + R25); and the
    chunked loop runs the FP32 kernel too (checked by replaying the oracle's PSO loop
    on the GPU's own J, as in test_gpu_forward_f32.py)."""
    import torch
    wl = wlm.scaled(wlm.config(0), n_iters=40)
    trace = oracle_trace(wl)
    full = orc.pso_invert(orc.model_from(wl), orc.box_from(wl),
                          orc.swarm_from(wl, async_chunk=24), 0, trace, wl["z0"], wl["v0"],
                          openmp=True)
    target, k = _cut_target(full["gbest_hist"][:, 0, 2], 10)
    g, o = _both(afm, wl, trace, seed=0, j_target=target, async_chunk=24)
    assert o["n_iters_done"] == k + 1 < 40
    _compare_cut_runs(g, o, 2)
    w32 = wlm.scaled(wlm.config(2), n_cycles=12, n_skip_cycles=6, n_particles=50, n_iters=5)
    tr = oracle_trace(w32)
    sw = afm.swarm_from(w32, async_chunk=16)
    g = afm.afm_pso_invert(afm.bounds_from(w32), sw, 4, torch.as_tensor(tr, device="cuda"),
                           afm.cfg_from(w32, precision=afm.F32), dump=True, hist=True)
    d = g["dump"].cpu().numpy()
    calls = {"k": 0}
    # evaluation order of the chunked swarm: batch, chunk, particle
    order = [(it, p) for it in range(5) for c0 in range(0, 50, 16)
             for p in range(c0, min(c0 + 16, 50))]

    def gpu_cost(theta, _U):
        it, p = order[calls["k"]]
        calls["k"] += 1
        return d[it, p, 9]

    o = orc.pso_core(gpu_cost, 3, orc.box_from(w32), orc.swarm_from(w32, async_chunk=16), 4, tr)
    assert calls["k"] == 250 and np.array_equal(o["dump"], d)
    assert np.array_equal(o["gbest_hist"], g["gbest_hist"].cpu().numpy())


def test_async_is_refused_where_it_has_no_meaning(afm):
    wl = wlm.scaled(wlm.config(0), n_particles=32, n_iters=2)
    sw = afm.swarm_from(wl, async_chunk=8)
    st = afm.afm_pso_init(afm.bounds_from(wl), afm.swarm_from(wl), 2, 1, 0)
    import torch
    J = torch.zeros(32, dtype=torch.float64, device="cuda")
    with pytest.raises(afm.AfmError) as e:
        afm.afm_pso_step(afm.bounds_from(wl), sw, 2, 1, 0, 0, True, J, st)
    assert e.value.code == afm.EUNSUPPORTED

"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py
times (default options), on sampled outputs the oracle can compute one by one
plus properties that hold at any size.

configs[1]: all 65 536 particles x 51 200 steps on the GPU, 160 sampled
particles through the oracle (FP64 1e-9; FP32 1e-3 with the c-15 protocol).
configs[2], [3], [4]: the full swarm for the first PSO batches; sampled
particles' misfits against the oracle at the positions the GPU evaluated, and
personal/global-best consistency over ALL particles.
"""
import numpy as np
import pytest

from oracle import binding as orc
from paper_1109_0334_b200 import workloads as wlm
from parity_helpers import oracle_trace, rel_err

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def afm():
    import torch
    assert torch.cuda.is_available()
    from paper_1109_0334_b200 import afm as m
    m.lib()
    for k in ("block", "tile", "ppt"):
        m.afm_set_option(k, 0)
    return m


@pytest.fixture(scope="module")
def cfg1_inputs():
    wl = wlm.config(1)
    P = wl["swarm"]["n_particles"]
    trace = oracle_trace(wl)
    params = wlm.draw_params(wl, P, seed=1)
    z0v0 = wlm.draw_initial_states(wl, P, seed=2)
    pick = np.random.default_rng(7).choice(P, size=160, replace=False)
    pick[:4] = [0, 31, P - 32, P - 1]          # first/last warp edges
    Jo = orc.forward_batch(orc.model_from(wl), params[pick], trace, z0v0=z0v0[pick],
                           openmp=True)
    return wl, trace, params, z0v0, pick, Jo


def _forward(afm, wl, params, trace, z0v0, precision):
    import torch
    J = afm.afm_forward_batch(torch.as_tensor(params, device="cuda"),
                              torch.as_tensor(trace, device="cuda"),
                              afm.cfg_from(wl, precision=precision),
                              z0v0=torch.as_tensor(z0v0, device="cuda"))
    torch.cuda.synchronize()
    return J.cpu().numpy()


def test_cfg1_full_size_f64(afm, cfg1_inputs):
    wl, trace, params, z0v0, pick, Jo = cfg1_inputs
    Jg = _forward(afm, wl, params, trace, z0v0, afm.F64)
    assert Jg.shape == (65536,) and not np.isnan(Jg).any()
    e = rel_err(Jg[pick], Jo)
    # c-15: a chaotic particle is excused only if the oracle itself moves by more
    # than the tolerance under a 1e-13 relative change of its initial state
    M = orc.model_from(wl)
    for i in np.flatnonzero(e >= 1e-9):
        p, z = params[pick[i]][None], z0v0[pick[i]][None]
        J2 = orc.forward_batch(M, p, trace, z0v0=z * (1 + 1e-13))[0]
        assert abs(J2 - Jo[i]) / Jo[i] > 1e-9, (int(pick[i]), e[i])
    assert np.percentile(e, 95) < 1e-9
    # whole-batch properties: every misfit positive; J >= the noise floor scale
    assert (Jg[np.isfinite(Jg)] > 0).all()


def test_cfg1_full_size_f32(afm, cfg1_inputs):
    wl, trace, params, z0v0, pick, Jo = cfg1_inputs
    Jg = _forward(afm, wl, params, trace, z0v0, afm.F32)
    J64 = _forward(afm, wl, params, trace, z0v0, afm.F64)
    e = rel_err(Jg[pick], Jo)
    M = orc.model_from(wl)
    ill = 0.25 * 1e-3 / 2.0 ** -23 * 1e-10
    for i in np.flatnonzero(e >= 1e-3):
        p, z = params[pick[i]][None], z0v0[pick[i]][None]
        J2 = orc.forward_batch(M, p, trace, z0v0=z * (1 + 1e-10))[0]
        assert abs(J2 - Jo[i]) / Jo[i] > ill, (int(pick[i]), e[i])
    assert np.percentile(e, 95) < 1e-3
    # over ALL 65 536 particles, against the FP64 kernel (itself checked above)
    ea = rel_err(Jg, J64)
    print("cfg1 f32 vs f64 kernel, all particles: median %.2e p99 %.2e p99.9 %.2e, "
          "%d above 1e-3" % (np.median(ea), np.percentile(ea, 99),
                              np.percentile(ea, 99.9), int((ea >= 1e-3).sum())))
    assert np.percentile(ea, 99) < 1e-4
    assert (ea >= 1e-3).mean() < 5e-3


def _full_swarm_batches(afm, ci, n_iters, n_sample, precision=0, n_traces=None):
    import torch
    wl = wlm.config(ci)
    over = dict(n_iters=n_iters)
    if n_traces is not None:
        over["n_traces"] = n_traces
    wl = wlm.scaled(wl, **over)
    truths = None if wl["truth"] is not None else wlm.pixel_truths(wl)
    trace = oracle_trace(wl, truths=truths)
    T, per, D = wl["n_traces"], wl["swarm"]["n_particles"], wl["n_params"]
    g = afm.afm_pso_invert(afm.bounds_from(wl), afm.swarm_from(wl), wl["pso_seed"],
                           torch.as_tensor(trace, device="cuda"),
                           afm.cfg_from(wl, precision=precision), dump=True, hist=True)
    d = g["dump"]                                  # device [it][PT][3D+2]
    # properties over ALL particles, on the device
    J, pbJ = d[:, :, 3 * D], d[:, :, 3 * D + 1]
    run_min = torch.cummin(torch.nan_to_num(J, nan=float("inf")), dim=0).values
    assert torch.equal(pbJ, run_min)               # personal best = running minimum
    gh = g["gbest_hist"]                           # [it][T][D+1]
    seg_min = pbJ.reshape(n_iters, T, per).min(dim=2).values
    assert torch.equal(gh[:, :, D], seg_min)       # global best = min over the swarm
    lo = torch.as_tensor(wl["bounds"]["lo"], device="cuda")
    hi = torch.as_tensor(wl["bounds"]["hi"], device="cuda")
    x = d[:, :, 0:D]
    assert bool(((x >= lo) & (x <= hi)).all())
    # sampled particles through the oracle at the positions the GPU evaluated
    rng = np.random.default_rng(11 + ci)
    pick = rng.choice(T * per, size=n_sample, replace=False)
    M = orc.model_from(wl)
    worst = 0.0
    for it in range(n_iters):
        xs = d[it, pick, 0:D].cpu().numpy()
        Jg = d[it, pick, 3 * D].cpu().numpy()
        th = wlm.theta_of_coords(wl, xs)
        for s in np.unique(pick // per):
            m = (pick // per) == s
            Jo = orc.forward_batch(M, th[m], trace[s], z0=wl["z0"], v0=wl["v0"],
                                   openmp=True)
            worst = max(worst, rel_err(Jg[m], Jo).max())
    return worst


def test_cfg2_full_swarm_first_batches(afm):
    assert _full_swarm_batches(afm, 2, n_iters=3, n_sample=96) < 1e-9


def test_cfg3_full_swarm_first_batches_f64(afm):
    assert _full_swarm_batches(afm, 3, n_iters=2, n_sample=64) < 1e-9


def test_cfg3_full_swarm_first_batches_f32(afm):
    # 64 samples x 2 batches: the bulk bound (p99.9 of the FP32 error is 8e-4)
    assert _full_swarm_batches(afm, 3, n_iters=2, n_sample=64, precision=1) < 2e-3


def test_cfg4_full_line_scan_first_batches(afm):
    """All 256 pixels x 4 096 particles = 1 048 576 concurrent particles."""
    assert _full_swarm_batches(afm, 4, n_iters=2, n_sample=96) < 1e-9

"""GPU parity for the paper's own sample models: Hooke, Eq. 11
(PAPER.md:260), and Kelvin-Voigt, Eq. 12, through the C ABI,
against the CPU oracle on the same seeded inputs.  Same bar as the config laws:
FP64 misfit 1e-9 relative, FP32 1e-3, swarm state replayed."""
import numpy as np
import pytest

from oracle import binding as orc
from paper_1109_0334_b200 import workloads as wlm
from parity_helpers import oracle_trace, rel_err

pytestmark = pytest.mark.gpu
NAMES = ["hooke", "kelvin_voigt"]


@pytest.fixture(scope="module")
def afm():
    import torch
    assert torch.cuda.is_available()
    from paper_1109_0334_b200 import afm as m
    m.lib()
    return m


def _params(wl, n, seed):
    p = wlm.draw_params(wl, n, seed=seed)
    p[0] = wl["truth"]
    p[1] = wl["bounds"]["lo"]            # k_s = 0 (and h or zeta at the lower bound)
    p[2] = wl["bounds"]["hi"]
    return p


def _gpu(afm, wl, params, trace, precision):
    import torch
    J = afm.afm_forward_batch(torch.as_tensor(params, device="cuda"),
                              torch.as_tensor(np.ascontiguousarray(trace), device="cuda"),
                              afm.cfg_from(wl, precision=precision))
    torch.cuda.synchronize()
    return J.cpu().numpy()


@pytest.mark.parametrize("name", NAMES)
def test_trajectory_matches_oracle(afm, name):
    wl = wlm.scaled(wlm.paper_law(name), n_cycles=20, n_skip_cycles=10)
    bad, zs, vs = orc.integrate(orc.model_from(wl), wl["truth"], wl["z0"], wl["v0"])
    assert bad == 0
    gz, gv = afm.afm_trajectory(wl["truth"], afm.cfg_from(wl), wl["z0"], wl["v0"])
    A0 = wl["cantilever"]["A0"]
    w = 2 * np.pi * wl["cantilever"]["f_drive"]
    assert np.max(np.abs(gz - zs)) / A0 < 1e-11
    assert np.max(np.abs(gv - vs)) / (A0 * w) < 1e-11
    # the tip really reaches the sample in this workload
    h = wl["truth"][1] if name == "hooke" else wl["cantilever"]["z_c"]
    assert zs.min() + h < -0.2e-9


@pytest.mark.parametrize("name", NAMES)
def test_forward_batch_f64(afm, name):
    wl = wlm.paper_law(name)                       # full length: 60 cycles x 256
    trace = oracle_trace(wl)
    params = _params(wl, 1031, seed=31)
    Jo = orc.forward_batch(orc.model_from(wl), params, trace, z0=wl["z0"], v0=wl["v0"],
                           openmp=True)
    Jg = _gpu(afm, wl, params, trace, afm.F64)
    assert np.all(np.isfinite(Jo))
    e = rel_err(Jg, Jo)
    assert e.max() < 1e-9, (e.max(), int(e.argmax()))
    # J(truth) on the noisy trace ~ W sigma^2
    assert Jg[0] == pytest.approx(wl["n_window"] * wl["sigma"] ** 2, rel=0.1)


@pytest.mark.parametrize("name", NAMES)
def test_forward_batch_f32(afm, name):
    wl = wlm.paper_law(name)
    trace = oracle_trace(wl)
    params = _params(wl, 1031, seed=32)
    M = orc.model_from(wl)
    Jo = orc.forward_batch(M, params, trace, z0=wl["z0"], v0=wl["v0"], openmp=True)
    Jg = _gpu(afm, wl, params, trace, afm.F32)
    e = rel_err(Jg, Jo)
    print("%s f32: median %.2e p99 %.2e max %.2e" % (name, np.median(e),
                                                     np.percentile(e, 99), e.max()))
    assert np.percentile(e, 99) < 1e-4
    # Above the tolerance only where the law itself is discontinuous within FP32's
    # reach.  Kelvin-Voigt's force JUMPS by -zeta v at touch: an RK4 stage point
    # that lands within the FP32 trajectory accuracy (~1e-6 nm at A0 = 10 nm) of
    # the surface takes the other branch -- for any FP32 scheme.  Criterion, from
    # the ORACLE's own trajectory: some stage point of the particle lies within
    # 2e-6 nm of the surface (typical particles: 1e-5..1e-4 nm).  Hooke is
    # continuous: no particle may exceed the tolerance.
    out = np.flatnonzero(e >= 1e-3)
    assert out.size <= (0 if name == "hooke" else 8), (out.size, e[out])
    for i in out:
        g = _min_stage_gap(M, wl, params[i])
        print("  outlier %d: err %.2e, nearest stage point %.2e nm from the surface"
              % (i, e[i], g * 1e9))
        assert g < 2e-15, (int(i), e[i], g)


def _min_stage_gap(M, wl, th):
    """Smallest |gap| over the RK4 stage points of the oracle's trajectory (the
    classical tableau restated with the oracle's own right-hand side)."""
    c = orc.constants(M)
    zc, dt = wl["cantilever"]["z_c"], c.dt
    bad, zs, vs = orc.integrate(M, th, wl["z0"], wl["v0"])
    g = zs + zc
    near = np.flatnonzero((np.abs(g[:-1]) < 0.5e-9) | (np.abs(g[1:]) < 0.5e-9))
    best = np.inf
    for n in near:
        t, z, v = n * dt, zs[n], vs[n]
        k1z, k1v = orc.rhs(M, th, t, z, v)
        p2, v2 = z + 0.5 * dt * k1z, v + 0.5 * dt * k1v
        k2z, k2v = orc.rhs(M, th, t + 0.5 * dt, p2, v2)
        p3, v3 = z + 0.5 * dt * k2z, v + 0.5 * dt * k2v
        k3z, _ = orc.rhs(M, th, t + 0.5 * dt, p3, v3)
        p4 = z + dt * k3z
        best = min(best, abs(z + zc), abs(p2 + zc), abs(p3 + zc), abs(p4 + zc))
    return best


@pytest.mark.parametrize("name", NAMES)
def test_inversion_replays_the_oracle(afm, name):
    import torch
    wl = wlm.scaled(wlm.paper_law(name), n_cycles=16, n_skip_cycles=8, n_particles=96,
                    n_iters=8)
    trace = oracle_trace(wl)
    g = afm.afm_pso_invert(afm.bounds_from(wl), afm.swarm_from(wl), wl["pso_seed"],
                           torch.as_tensor(trace, device="cuda"), afm.cfg_from(wl),
                           dump=True)
    o = orc.pso_invert(orc.model_from(wl), orc.box_from(wl), orc.swarm_from(wl),
                       wl["pso_seed"], trace, wl["z0"], wl["v0"], dump=True, openmp=True)
    gd, od = g["dump"].cpu().numpy(), o["dump"]
    D = 2
    scale = np.array(wl["bounds"]["hi"])
    assert np.max(np.abs(gd[..., 0:D] - od[..., 0:D]) / scale) < 1e-9      # x
    assert rel_err(gd[..., 3 * D], od[..., 3 * D]).max() < 1e-9            # J
    assert rel_err(g["J_star"], o["J_star"]).max() < 1e-9
    assert np.max(np.abs(g["theta_star"] - o["theta_star"]) / scale) < 1e-9


@pytest.mark.parametrize("name", NAMES)
def test_full_inversion_recovers_the_truth_noise_free(afm, name):
    """The paper's experiment (Figs. 10, 11) on the full workload: 1 024 particles x
    60 batches on a noise-free trace of the truth."""
    import torch
    wl = wlm.paper_law(name)
    trace = oracle_trace(wl, noise=False)
    g = afm.afm_pso_invert(afm.bounds_from(wl), afm.swarm_from(wl), wl["pso_seed"],
                           torch.as_tensor(trace, device="cuda"), afm.cfg_from(wl))
    rel = np.abs(g["theta_star"][0] - np.array(wl["truth"])) / np.array(wl["truth"])
    print(name, "theta* rel err", rel, "J*", g["J_star"])
    # Kelvin-Voigt's cost landscape is corrugated: after 60 batches
    # the swarm is within 0.2 % of the truth and still contracting
    assert rel.max() < (1e-3 if name == "hooke" else 5e-3)

"""GPU parity for the multi-mode Euler-Bernoulli forward model (the paper's own
forward problem) through the C ABI against the CPU oracle:
initialisation data (Newton roots, Simpson inner products), trajectories,
forward-batch misfits (1e-9 relative), swarm replay."""
import math

import numpy as np
import pytest

from oracle import binding as orc
from paper_1109_0334_b200 import workloads as wlm
from parity_helpers import rel_err

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def afm():
    import torch
    assert torch.cuda.is_available()
    from paper_1109_0334_b200 import afm as m
    m.lib()
    return m


def _trace(wl, B, noise=True):
    bad, win = orc.beam_window(B, wl["truth"])
    assert bad == 0
    tr = win[None, :]
    return tr + wlm.trace_noise(wl) if noise else tr


def test_initialisation_kernel_matches_oracle_and_appendix_a(afm):
    wl = wlm.beam_workload()
    g = afm.afm_beam_modes(afm.beam_cfg_from(wl))
    mo = orc.beam_setup(orc.beam_from(wl))
    for i in range(8):
        assert g["beta_L"][i] == pytest.approx(mo.bL[i], rel=1e-14)
        assert g["omega"][i] == pytest.approx(mo.omega[i], rel=1e-13)
        assert g["phi_L"][i] == pytest.approx(mo.phiL[i], rel=1e-12)
        assert g["participation"][i] == pytest.approx(mo.phiL[i] * mo.intphi[i] / mo.norm[i],
                                                      rel=1e-11)
        assert g["compliance"][i] == pytest.approx(mo.phiL[i] * mo.fgain[i], rel=1e-11)
    assert g["omega"][0] / (2 * math.pi) == pytest.approx(25468.9, abs=0.05)


@pytest.mark.parametrize("law,n_modes", [(wlm.LAW_NONE, 8), (wlm.LAW_DMT, 8), (wlm.LAW_DMT, 1),
                                         (wlm.LAW_DMT, 4), (wlm.LAW_DMT_VISC, 2),
                                         (wlm.LAW_KELVIN_VOIGT, 8), (wlm.LAW_LJ_EXP, 8)])
def test_trajectory_matches_oracle(afm, law, n_modes):
    wl = wlm.scaled(wlm.beam_workload(), n_cycles=40, n_skip_cycles=20)
    theta = {wlm.LAW_NONE: [], wlm.LAW_DMT: [1e-19, 1e9], wlm.LAW_DMT_VISC: [1e-19, 1e9, 100.0],
             wlm.LAW_KELVIN_VOIGT: [4.0, 5e-6],
             wlm.LAW_LJ_EXP: [1e-81, 1.667e-28, 1e-9, 1e-9]}[law]
    wl = dict(wl, law=law, n_params=len(theta), beam=dict(wl["beam"], n_modes=n_modes))
    if law == wlm.LAW_LJ_EXP:
        wl["beam"]["z_c"] = 10.5e-9
    B = orc.beam_from(wl)
    bad, u, v, _ = orc.beam_integrate(B, theta + [0.0] * (4 - len(theta)))
    assert bad == 0
    gu, gv = afm.afm_beam_trajectory(theta + [0.0] * (4 - len(theta)), afm.beam_cfg_from(wl))
    A, w = wl["beam"]["A_ref"], 2 * math.pi * wl["beam"]["f_drive"]
    assert np.max(np.abs(gu - u)) / A < 1e-10
    assert np.max(np.abs(gv - v)) / (A * w) < 1e-9      # stiff modes dominate the tip velocity
    if law in (wlm.LAW_DMT, wlm.LAW_DMT_VISC):
        assert u.min() + wl["beam"]["z_c"] < wl["beam"]["a0"]     # the tip taps


def test_forward_batch_full_length(afm):
    """The whole workload length (80 cycles x 512 steps, 8 modes) on 515 particles
    (ragged CTAs): per-particle misfit within 1e-9 of the oracle."""
    import torch
    wl = wlm.beam_workload()
    B = orc.beam_from(wl)
    trace = _trace(wl, B)
    params = wlm.draw_params(wl, 515, seed=41)
    params[0] = wl["truth"]
    Jo = orc.beam_forward_batch(B, params, trace, openmp=True)
    J = afm.afm_beam_forward_batch(torch.as_tensor(params, device="cuda"),
                                   torch.as_tensor(trace, device="cuda"),
                                   afm.beam_cfg_from(wl))
    torch.cuda.synchronize()
    Jg = J.cpu().numpy()
    assert np.all(np.isfinite(Jo))
    e = rel_err(Jg, Jo)
    print("beam f64: median %.2e max %.2e" % (np.median(e), e.max()))
    assert e.max() < 1e-9, (e.max(), int(e.argmax()))
    assert Jg[0] == pytest.approx(wl["n_window"] * wl["sigma"] ** 2, rel=0.1)
    # coordinates in (bounds given) == physical parameters in
    coords = wlm.draw_coords(wl, 515, seed=41)
    coords[0] = np.log10(wl["truth"])
    Jc = afm.afm_beam_forward_batch(torch.as_tensor(coords, device="cuda"),
                                    torch.as_tensor(trace, device="cuda"),
                                    afm.beam_cfg_from(wl), bounds=afm.bounds_from(wl))
    torch.cuda.synchronize()
    assert rel_err(Jc.cpu().numpy()[1:], Jg[1:]).max() < 1e-9


def test_forward_batch_traces_modes_and_divergence(afm):
    import torch
    wl = wlm.scaled(wlm.beam_workload(), n_cycles=36, n_skip_cycles=18, n_traces=3)
    wl = dict(wl, beam=dict(wl["beam"], n_modes=4))
    B = orc.beam_from(wl)
    truths = wlm.theta_of_coords(wl, wlm.draw_coords(wl, 3, seed=5))
    trace = np.stack([orc.beam_window(B, t)[1] for t in truths]) + wlm.trace_noise(wl)
    params = wlm.draw_params(wl, 3 * 45, seed=42)
    Jo = orc.beam_forward_batch(B, params, trace, n_traces=3, openmp=True)
    J = afm.afm_beam_forward_batch(torch.as_tensor(params, device="cuda"),
                                   torch.as_tensor(trace, device="cuda"),
                                   afm.beam_cfg_from(wl))
    torch.cuda.synchronize()
    assert rel_err(J.cpu().numpy(), Jo).max() < 1e-9
    # divergence rule: a tiny reference amplitude makes every trajectory "run away"
    wd = dict(wl, beam=dict(wl["beam"], A_ref=1e-11))
    Jd = afm.afm_beam_forward_batch(torch.as_tensor(params, device="cuda"),
                                    torch.as_tensor(trace, device="cuda"),
                                    afm.beam_cfg_from(wd))
    torch.cuda.synchronize()
    assert np.isinf(Jd.cpu().numpy()).all()
    assert np.isinf(orc.beam_forward_batch(orc.beam_from(wd), params[:4], trace[:1],
                                           n_traces=1)).all()


def test_inversion_replays_the_oracle_and_recovers_the_truth(afm):
    import torch
    wl = wlm.scaled(wlm.beam_workload(), n_cycles=40, n_skip_cycles=20, n_particles=64,
                    n_iters=6)
    B = orc.beam_from(wl)
    trace = _trace(wl, B)
    g = afm.afm_beam_pso_invert(afm.bounds_from(wl), afm.swarm_from(wl), wl["pso_seed"],
                                torch.as_tensor(trace, device="cuda"),
                                afm.beam_cfg_from(wl), dump=True, hist=True)
    o = orc.beam_pso_invert(B, orc.box_from(wl), orc.swarm_from(wl), wl["pso_seed"], trace,
                            dump=True, openmp=True)
    gd, od = g["dump"].cpu().numpy(), o["dump"]
    assert np.max(np.abs(gd[..., 0:2] - od[..., 0:2])) < 1e-9          # x (log10 coordinates)
    assert rel_err(gd[..., 6], od[..., 6]).max() < 1e-9                # J
    assert rel_err(gd[..., 7], od[..., 7]).max() < 1e-9                # pbestJ
    assert rel_err(g["J_star"], o["J_star"]).max() < 1e-9
    assert rel_err(g["theta_star"], o["theta_star"]).max() < 1e-9
    # the full workload on a noise-free trace: 1 024 particles x 40 batches
    wf = wlm.beam_workload()
    clean = _trace(wf, orc.beam_from(wf), noise=False)
    r = afm.afm_beam_pso_invert(afm.bounds_from(wf), afm.swarm_from(wf), wf["pso_seed"],
                                torch.as_tensor(clean, device="cuda"), afm.beam_cfg_from(wf))
    rel = np.abs(r["theta_star"][0] - np.array(wf["truth"])) / np.array(wf["truth"])
    print("beam inversion theta* rel err", rel, "J*", r["J_star"])
    assert rel.max() < 1e-2


@pytest.mark.parametrize("segs,workers,n_modes", [(0, 0, 8), (5, 1, 8), (36, 3, 4), (2, 8, 2)])
def test_segment_queue_changes_no_beam_result(afm, segs, workers, n_modes):
    """beam_integrate_f64_q (persistent workers, priority queue of time segments, the
    modal state of a chain checkpointed between segments) against the one-CTA-per-warp
    kernel: misfits of a ragged multi-trace batch and the swarm of a short inversion
    must be bit-identical; (5, 1): 626 chains on 592 workers, so chains wait."""
    import torch
    wl = wlm.scaled(wlm.beam_workload(), n_cycles=36, n_skip_cycles=18, n_traces=3,
                    n_particles=77, n_iters=3)
    wl = dict(wl, beam=dict(wl["beam"], n_modes=n_modes))
    B = orc.beam_from(wl)
    truths = wlm.theta_of_coords(wl, wlm.draw_coords(wl, 3, seed=5))
    trace = np.stack([orc.beam_window(B, t)[1] for t in truths]) + wlm.trace_noise(wl)
    n = 3 * 6677 if workers == 1 else 3 * 313
    params = wlm.draw_params(wl, n, seed=42)
    cfg = afm.beam_cfg_from(wl)
    t = torch.as_tensor(trace, device="cuda")
    out = {}
    for queue in (1, 2):
        afm.afm_set_option("queue", queue)
        afm.afm_set_option("segs", segs)
        afm.afm_set_option("workers", workers)
        try:
            J = afm.afm_beam_forward_batch(torch.as_tensor(params, device="cuda"), t, cfg)
            g = afm.afm_beam_pso_invert(afm.bounds_from(wl), afm.swarm_from(wl), 3, t, cfg,
                                        dump=True)
            torch.cuda.synchronize()
            out[queue] = (J.cpu().numpy(), g["dump"].cpu().numpy(), g["theta_star"])
        finally:
            for name in ("queue", "segs", "workers"):
                afm.afm_set_option(name, 0)
    for a, b in zip(out[1], out[2]):
        assert np.array_equal(a, b)
    pick = np.arange(0, n, 97)
    # the oracle on a sample of the batch (trace of each sampled particle's segment)
    per = n // 3
    for s in range(3):
        idx = pick[(pick >= s * per) & (pick < (s + 1) * per)]
        Jo = orc.beam_forward_batch(B, params[idx], trace[s:s + 1], n_traces=1, openmp=True)
        assert rel_err(out[2][0][idx], Jo).max() < 1e-9


def test_full_size_batch_as_benched(afm):
    """The batch bench.py --one-batch 7 times (65 536 particles x 40 960 steps x 8
    modes, default options: the segment-queue kernel with 3 workers per
    sub-partition): every 512th particle against the oracle at 1e-9, every misfit
    finite, and the plain kernel gives the same bits."""
    import torch
    wl = wlm.beam_workload()
    B = orc.beam_from(wl)
    trace = _trace(wl, B)
    n = 65536
    params = wlm.draw_params(wl, n, seed=1)
    cfg = afm.beam_cfg_from(wl)
    t = torch.as_tensor(trace, device="cuda")
    p = torch.as_tensor(params, device="cuda")
    J = afm.afm_beam_forward_batch(p, t, cfg)
    afm.afm_set_option("queue", 1)
    try:
        Jp = afm.afm_beam_forward_batch(p, t, cfg)
        torch.cuda.synchronize()
    finally:
        afm.afm_set_option("queue", 0)
    assert torch.equal(J, Jp)
    Jg = J.cpu().numpy()
    assert np.all(np.isfinite(Jg))
    pick = np.arange(0, n, 512)
    Jo = orc.beam_forward_batch(B, params[pick], trace, openmp=True)
    e = rel_err(Jg[pick], Jo)
    print("beam full size: median %.2e max %.2e" % (np.median(e), e.max()))
    assert e.max() < 1e-9, (e.max(), int(e.argmax()))

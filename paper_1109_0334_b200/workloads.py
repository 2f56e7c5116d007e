"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is the ONLY code shared by the CPU oracle and the CUDA
path: it holds workload constants and seeded random draws, and none of the
method's arithmetic (no ODE, no force law, no misfit, no PSO).  It imports
neither of them.  numpy only.

The paper measures on no public dataset: its workloads are synthetic
deflection traces made by its own CPU solver.  The five
configs below stand in for them.

Units: SI throughout.  PSO coordinates x: theta_j = 10**x_j where
bounds["log10"][j] is 1, else theta_j = x_j.
"""
import math

import numpy as np

LAW_NONE, LAW_DMT, LAW_DMT_VISC, LAW_LJ_EXP, LAW_HOOKE, LAW_KELVIN_VOIGT = 0, 1, 2, 3, 4, 5

_PSO = dict(w=0.72, c1=1.49, c2=1.49)   # BASELINE.json configs[0]


def _free_steady_state(c):
    """Initial state ON the free steady-state orbit z(t) = A0 cos(w t - phi),
    tan(phi) = (r/Q)/(1-r^2) (reading R6).  An input choice: the
    closed-form orbit of the linear oscillator, not part of the method."""
    r = c["f_drive"] / c["f0"]
    phi = math.atan2(r / c["Q"], 1.0 - r * r)
    w = 2.0 * math.pi * c["f_drive"]
    if c["f_drive"] == c["f0"]:
        return 0.0, c["A0"] * w
    return c["A0"] * math.cos(phi), c["A0"] * w * math.sin(phi)


def _soft_cantilever():
    # configs[0]: k=2 N/m, f0=70 kHz, Q=100, drive at f0, A0=10 nm, z_c=8 nm,
    # R=10 nm, a0=0.3 nm
    return dict(k=2.0, f0=70e3, Q=100.0, f_drive=70e3, A0=10e-9, z_c=8e-9,
                R=10e-9, a0=0.3e-9)


def _stiff_cantilever():
    # configs[3]: k=40 N/m, f0=300 kHz, Q=400, A0=20 nm; z_c is not given by
    # BASELINE.json: 20.5 nm per DESIGN.md reading R9.  R, a0 unused by LJ+exp.
    return dict(k=40.0, f0=300e3, Q=400.0, f_drive=300e3, A0=20e-9,
                z_c=20.5e-9, R=10e-9, a0=0.3e-9)


def config(i):
    """Workload dict for BASELINE.json configs[i]."""
    if i == 0:
        wl = dict(name="cfg0_tiny_dmt_inversion", cantilever=_soft_cantilever(),
                  law=LAW_DMT, n_params=2, steps_per_cycle=100, n_cycles=20,
                  n_skip_cycles=10, sigma=0.05e-9,
                  truth=[1e-19, 1e9],
                  bounds=dict(lo=[-20.0, 8.0], hi=[-18.0, 10.0], log10=[1, 1]),
                  swarm=dict(n_particles=64, n_iters=20, **_PSO),
                  n_traces=1, precisions=["f64"])
    elif i == 1:
        wl = dict(name="cfg1_forward_batch_dmt", cantilever=_soft_cantilever(),
                  law=LAW_DMT, n_params=2, steps_per_cycle=256, n_cycles=200,
                  n_skip_cycles=100, sigma=0.05e-9,
                  truth=[1e-19, 1e9],
                  bounds=dict(lo=[-20.0, 8.0], hi=[-18.0, 10.0], log10=[1, 1]),
                  swarm=dict(n_particles=65536, n_iters=1, **_PSO),
                  n_traces=1, precisions=["f64", "f32"])
    elif i == 2:
        wl = dict(name="cfg2_dmt_visc_inversion", cantilever=_soft_cantilever(),
                  law=LAW_DMT_VISC, n_params=3, steps_per_cycle=256,
                  n_cycles=100, n_skip_cycles=50, sigma=0.02e-9,
                  truth=[1e-19, 1e9, 100.0],
                  bounds=dict(lo=[-20.0, 8.0, 1.0], hi=[-18.0, 10.0, 1000.0],
                              log10=[1, 1, 0]),
                  swarm=dict(n_particles=1024, n_iters=200, **_PSO),
                  n_traces=1, precisions=["f64"])
    elif i == 3:
        # ground truth per DESIGN.md reading R9 (BASELINE.json gives none)
        truth = [1e-81, 1.0e-19 * 10e-9 / 6.0, 1e-9, 1e-9]
        lo = [math.log10(t) - 1.0 for t in truth]
        hi = [math.log10(t) + 1.0 for t in truth]
        wl = dict(name="cfg3_lj_exp_inversion", cantilever=_stiff_cantilever(),
                  law=LAW_LJ_EXP, n_params=4, steps_per_cycle=512,
                  n_cycles=150, n_skip_cycles=75, sigma=0.01e-9,
                  truth=truth,
                  bounds=dict(lo=lo, hi=hi, log10=[1, 1, 1, 1]),
                  swarm=dict(n_particles=8192, n_iters=300, **_PSO),
                  n_traces=1, precisions=["f32", "f64"])
    elif i == 4:
        wl = dict(name="cfg4_line_scan", cantilever=_soft_cantilever(),
                  law=LAW_DMT_VISC, n_params=3, steps_per_cycle=256,
                  n_cycles=50, n_skip_cycles=25, sigma=0.02e-9,
                  truth=None,   # per pixel: see pixel_truths()
                  bounds=dict(lo=[-20.0, 8.0, 1.0], hi=[-18.0, 10.0, 1000.0],
                              log10=[1, 1, 0]),
                  swarm=dict(n_particles=4096, n_iters=100, **_PSO),
                  n_traces=256, precisions=["f64"])
    else:
        raise ValueError("configs are 0..4")
    wl["index"] = i
    wl["pso_seed"] = 0
    wl["trace_seed"] = 1000 + i
    wl["z0"], wl["v0"] = _free_steady_state(wl["cantilever"])
    wl["n_steps"] = wl["steps_per_cycle"] * wl["n_cycles"]
    wl["n_window"] = wl["steps_per_cycle"] * (wl["n_cycles"] - wl["n_skip_cycles"])
    return wl


def paper_law(name):
    """The paper's own two sample models as extra workloads,
    on the configs[0] cantilever.  Index 5 = "hooke" (Eq. 11, PAPER.md:260:
    unknowns k_s and the separation h), 6 = "kelvin_voigt" (Eq. 12,
    PAPER.md:270: unknowns k_s and zeta_s, separation known).  The paper's truth
    k_s = 4 N/m and its search range [0, 25] N/m are kept; its h = 50 nm and
    zeta_s = 0.1 N s/m belong to its own cantilever and step (at this one,
    zeta_s h/m = 541 per step is far outside RK4's stability region), so h is
    scaled with the amplitude (8 nm at A0 = 10 nm) and zeta_s to 5e-6 N s/m
    (range [0, 2e-5]).  DESIGN.md readings R19/R20.  All coordinates linear."""
    if name == "hooke":
        wl = dict(name="paper_hooke_inversion", cantilever=_soft_cantilever(),
                  law=LAW_HOOKE, n_params=2, steps_per_cycle=256, n_cycles=60,
                  n_skip_cycles=30, sigma=0.02e-9, truth=[4.0, 8e-9],
                  bounds=dict(lo=[0.0, 5e-9], hi=[25.0, 11e-9], log10=[0, 0]),
                  swarm=dict(n_particles=1024, n_iters=60, **_PSO),
                  n_traces=1, precisions=["f64", "f32"], index=5)
    elif name == "kelvin_voigt":
        wl = dict(name="paper_kelvin_voigt_inversion", cantilever=_soft_cantilever(),
                  law=LAW_KELVIN_VOIGT, n_params=2, steps_per_cycle=256, n_cycles=60,
                  n_skip_cycles=30, sigma=0.02e-9, truth=[4.0, 5e-6],
                  bounds=dict(lo=[0.0, 0.0], hi=[25.0, 2e-5], log10=[0, 0]),
                  swarm=dict(n_particles=1024, n_iters=60, **_PSO),
                  n_traces=1, precisions=["f64", "f32"], index=6)
    else:
        raise ValueError('paper_law: "hooke" or "kelvin_voigt"')
    wl["pso_seed"] = 0
    wl["trace_seed"] = 1000 + wl["index"]
    wl["z0"], wl["v0"] = _free_steady_state(wl["cantilever"])
    wl["n_steps"] = wl["steps_per_cycle"] * wl["n_cycles"]
    wl["n_window"] = wl["steps_per_cycle"] * (wl["n_cycles"] - wl["n_skip_cycles"])
    return wl


def beam_workload():
    """The paper's own forward model as an extra workload: the
    Appendix A cantilever (L = 525 um, E = 1.76e11 Pa, 35 x 5 um
    section, mu = 4.0775e-7 kg/m, 8 modes, 501 modal-function points; first
    natural frequency 25 468.9 Hz), base-excited at that frequency, tapping on a
    DMT sample.  The paper gives no damping and no tapping set-point: Q = 50 and
    a base amplitude that makes the free tip amplitude ~10 nm (A_base = A_ref /
    (1.566 Q), 1.566 = first-mode participation factor) with the sample 8 nm
    below the tip (R21).  S = 512 steps per cycle keeps RK4 stable on
    mode 8 (h w_8 = 1.94); starts from rest, 80 cycles, misfit over the last 40."""
    width, height = 35e-6, 5e-6
    beam = dict(L=525e-6, E=1.76e11, I=width * height ** 3 / 12.0, mu=4.0775e-7,
                Q=50.0, f_drive=25468.9, A_ref=10e-9, A_base=10e-9 / (1.566 * 50.0),
                z_c=8e-9, R=10e-9, a0=0.3e-9, n_modes=8, n_points=501)
    wl = dict(name="paper_beam_dmt_inversion", beam=beam, law=LAW_DMT, n_params=2,
              steps_per_cycle=512, n_cycles=80, n_skip_cycles=40, sigma=0.02e-9,
              truth=[1e-19, 1e9],
              bounds=dict(lo=[-20.0, 8.0], hi=[-18.0, 10.0], log10=[1, 1]),
              swarm=dict(n_particles=1024, n_iters=40, **_PSO),
              n_traces=1, precisions=["f64"], index=7, pso_seed=0, trace_seed=1007)
    wl["n_steps"] = wl["steps_per_cycle"] * wl["n_cycles"]
    wl["n_window"] = wl["steps_per_cycle"] * (wl["n_cycles"] - wl["n_skip_cycles"])
    return wl


def _rng(seed):
    return np.random.Generator(np.random.Philox(key=int(seed)))


def theta_of_coords(wl, x):
    """Physical parameters of PSO coordinates (inputs only: used to draw
    log-uniform parameter sets, never by either implementation's PSO)."""
    x = np.asarray(x, dtype=np.float64)
    lg = np.asarray(wl["bounds"]["log10"], dtype=bool)
    return np.where(lg, np.power(10.0, np.where(lg, x, 0.0)), x)


def draw_coords(wl, n, seed):
    """n points uniform in the PSO-coordinate box, [n][D]."""
    lo = np.asarray(wl["bounds"]["lo"])
    hi = np.asarray(wl["bounds"]["hi"])
    u = _rng(seed).random((n, wl["n_params"]))
    return lo + u * (hi - lo)


def draw_params(wl, n, seed=1):
    """n parameter sets uniform in the coordinates (log-uniform where the
    coordinate is log10), [n][D] physical SI (configs[1])."""
    return theta_of_coords(wl, draw_coords(wl, n, seed))


def draw_initial_states(wl, n, seed=2):
    """configs[1]: z0 = A0 cos(phi0), phi0 ~ U[0, 2pi); v0 = -A0 w sin(phi0)
    (reading R6).  Returns [n][2]."""
    c = wl["cantilever"]
    phi0 = 2.0 * math.pi * _rng(seed).random(n)
    w = 2.0 * math.pi * c["f_drive"]
    return np.stack([c["A0"] * np.cos(phi0), -c["A0"] * w * np.sin(phi0)], axis=1)


def pixel_truths(wl, seed=None):
    """configs[4]: one ground truth per pixel, uniform within the bounds in
    PSO coordinates.  [n_traces][D] physical SI."""
    seed = wl["trace_seed"] + 7 if seed is None else seed
    return theta_of_coords(wl, draw_coords(wl, wl["n_traces"], seed))


def trace_noise(wl, n_traces=None, seed=None):
    """sigma * N(0,1), [n_traces][W]: the measurement noise added to the clean
    window of the ground-truth trajectory (whoever integrates it)."""
    n_traces = wl["n_traces"] if n_traces is None else n_traces
    seed = wl["trace_seed"] if seed is None else seed
    return wl["sigma"] * _rng(seed).standard_normal((n_traces, wl["n_window"]))


def scaled(wl, **kw):
    """Copy of a workload with some sizes overridden (parity-test subsamples):
    n_cycles, n_skip_cycles, steps_per_cycle, n_particles, n_iters, n_traces."""
    out = dict(wl)
    out["swarm"] = dict(wl["swarm"])
    for k, v in kw.items():
        if k in ("n_particles", "n_iters"):
            out["swarm"][k] = v
        else:
            out[k] = v
    out["n_steps"] = out["steps_per_cycle"] * out["n_cycles"]
    out["n_window"] = out["steps_per_cycle"] * (out["n_cycles"] - out["n_skip_cycles"])
    return out

"""Pins for the oracle's nonlinear forward solve: an adaptive library
integrator (scipy DOP853) on the same ODE written independently in numpy,
energy balance per cycle, and misfit identities (Eq. 5)."""
import math

import numpy as np
import pytest
from scipy.integrate import solve_ivp

from oracle import binding as orc
from paper_1109_0334_b200 import workloads as wlm


# --- the ODE typed independently of oracle/ (numpy / math only) -------------

def _numpy_rhs(wl, theta):
    c = wl["cantilever"]
    w0 = 2 * math.pi * c["f0"]
    w = 2 * math.pi * c["f_drive"]
    m = c["k"] / w0 ** 2
    r = w / w0
    F0 = c["k"] * c["A0"] * math.hypot(1 - r * r, r / c["Q"])
    law = wl["law"]

    def fts(d, v):
        if law == wlm.LAW_LJ_EXP:
            return theta[0] * d ** -8 - theta[1] * d ** -2 - theta[2] * math.exp(-d / theta[3])
        if d > c["a0"]:
            return -theta[0] * c["R"] / (6 * d ** 2)
        dl = c["a0"] - d
        f = -theta[0] * c["R"] / (6 * c["a0"] ** 2) + 4 / 3 * theta[1] * math.sqrt(c["R"]) * dl ** 1.5
        if law == wlm.LAW_DMT_VISC:
            f -= theta[2] * math.sqrt(c["R"] * dl) * v
        return f

    def f(t, y):
        z, v = y
        return [v, (F0 * math.cos(w * t) - m * w0 / c["Q"] * v - c["k"] * z + fts(z + c["z_c"], v)) / m]
    return f


def _scipy_reference(wl, theta, n_cycles):
    T = n_cycles / wl["cantilever"]["f_drive"]
    # scale to nm / (nm per unit time) inside the tolerance by using tiny atol
    sol = solve_ivp(_numpy_rhs(wl, theta), (0.0, T), [wl["z0"], wl["v0"]], method="DOP853",
                    rtol=1e-12, atol=[1e-22, 1e-16], dense_output=True, max_step=T / (n_cycles * 64))
    return sol


def test_lj_exp_converges_at_fourth_order_to_scipy_dop853():
    """Smooth force law: error vs the adaptive reference falls ~16x per step halving."""
    wl = wlm.config(3)
    ncyc = 4
    sol = _scipy_reference(wl, wl["truth"], ncyc)
    errs = []
    for S in (256, 512, 1024):
        M = orc.model_from(wl, n_cycles=ncyc, S=S, n_skip=0)
        c = orc.constants(M)
        bad, zs, vs = orc.integrate(M, wl["truth"], wl["z0"], wl["v0"])
        assert bad == 0
        t = np.arange(c.N + 1) * c.dt
        errs.append(np.max(np.abs(zs - sol.sol(t)[0])))
    A0 = wl["cantilever"]["A0"]
    assert errs[0] < 1e-4 * A0
    # the wall (1/d^8) is steep, so the asymptotic regime starts late: demand order >= ~3.5
    assert errs[0] / errs[1] > 11 and errs[1] / errs[2] > 11, errs


@pytest.mark.parametrize("idx", [0, 2])
def test_dmt_laws_agree_with_scipy_dop853(idx):
    """DMT is only C^0 in its slope at d = a0 (the vdW branch arrives with
    slope H R/(3 a0^3) = 12 N/m, the contact branch leaves with 0), so fixed-step
    RK4 loses its order at each contact crossing; the error must still shrink
    with the step and be small at the configs' own step (S = 256)."""
    wl = wlm.config(idx)
    ncyc = 3
    sol = _scipy_reference(wl, wl["truth"], ncyc)
    errs = []
    for S in (128, 256, 1024):
        M = orc.model_from(wl, n_cycles=ncyc, S=S, n_skip=0)
        c = orc.constants(M)
        bad, zs, vs = orc.integrate(M, wl["truth"], wl["z0"], wl["v0"])
        assert bad == 0
        t = np.arange(c.N + 1) * c.dt
        errs.append(np.max(np.abs(zs - sol.sol(t)[0])))
        # the tip really does touch the sample in this window
        assert np.min(zs) + wl["cantilever"]["z_c"] < wl["cantilever"]["a0"]
    A0 = wl["cantilever"]["A0"]
    assert errs[1] < 2e-4 * A0, errs
    assert errs[1] < 0.5 * errs[0] and errs[2] < 0.3 * errs[1], errs


def _cycle_integrals(wl, theta, n_cycles, S=512):
    """Per-cycle work integrals over the LAST cycle from the oracle's own output
    (periodic trapezoid = rectangle rule over one period)."""
    M = orc.model_from(wl, n_cycles=n_cycles, S=S, n_skip=0)
    c = orc.constants(M)
    bad, zs, vs = orc.integrate(M, theta, wl["z0"], wl["v0"])
    assert bad == 0
    z, v = zs[-S:], vs[-S:]
    n = np.arange(c.N - S + 1, c.N + 1)
    drive = c.F0 * np.cos(2 * math.pi * n / S)
    E_in = np.sum(drive * v) * c.dt
    E_damp = np.sum(c.c * v * v) * c.dt
    return M, c, z, v, E_in, E_damp


def test_energy_balance_conservative_dmt():
    """Steady state, conservative tip force: drive work = cantilever damping
    loss per cycle; first-harmonic form sin(phi) = A/A0 (Cleveland et al.,
    ref [10] of the paper)."""
    wl = wlm.config(1)
    S = 512
    M, c, z, v, E_in, E_damp = _cycle_integrals(wl, wl["truth"], 400, S)
    assert E_in > 0
    assert E_in == pytest.approx(E_damp, rel=2e-4, abs=0.0)
    n = np.arange(c.N - S + 1, c.N + 1)
    ph = 2 * math.pi * n / S
    a = 2 / S * np.sum(z * np.cos(ph))
    b = 2 / S * np.sum(z * np.sin(ph))
    A = math.hypot(a, b)
    sinphi = b / A                   # z ~ A cos(w t - phi) => sin component = A sin(phi)
    assert 0.5 * M.A0 < A < 0.95 * M.A0        # tapping reduces the amplitude
    assert sinphi == pytest.approx(A / M.A0, rel=2e-3, abs=0.0)


def test_energy_balance_viscoelastic():
    """DMT + contact damping: drive work - cantilever damping = work dissipated
    by the -eta sqrt(R delta) v term, evaluated independently in numpy."""
    wl = wlm.config(2)
    S = 1024
    theta = [1e-19, 1e9, 200.0]   # (eta = 300 settles on the non-contact branch)
    M, c, z, v, E_in, E_damp = _cycle_integrals(wl, theta, 400, S)
    cl = wl["cantilever"]
    delta = np.maximum(cl["a0"] - (z + cl["z_c"]), 0.0)
    E_visc = np.sum(theta[2] * np.sqrt(cl["R"] * delta) * v * v) * c.dt
    assert E_visc > 0.02 * E_damp              # the term matters
    assert E_in - E_damp == pytest.approx(E_visc, rel=5e-3, abs=0.0)
    assert E_in > E_damp


# --- misfit identities --------------------------------------------------------

def test_misfit_zero_on_own_clean_window_and_equals_noise_energy():
    wl = wlm.config(0)
    M = orc.model_from(wl)
    bad, clean = orc.window(M, wl["truth"], wl["z0"], wl["v0"])
    assert bad == 0
    assert orc.misfit(M, wl["truth"], wl["z0"], wl["v0"], clean) == 0.0
    noise = wlm.trace_noise(wl)[0]
    J = orc.misfit(M, wl["truth"], wl["z0"], wl["v0"], clean + noise)
    assert J == pytest.approx(np.sum(noise ** 2), rel=1e-6, abs=0.0)
    # chi-square scale: W sigma^2 +- a few sqrt(2W) sigma^2
    W, s2 = wl["n_window"], wl["sigma"] ** 2
    assert abs(J - W * s2) < 5 * math.sqrt(2 * W) * s2


def test_window_and_misfit_indexing_by_brute_force():
    """J = sum_{n=N-W+1}^{N} (z_n - U_{n-(N-W)-1})^2 over post-step states."""
    wl = wlm.scaled(wlm.config(0), n_cycles=6, n_skip_cycles=4, steps_per_cycle=50)
    M = orc.model_from(wl)
    c = orc.constants(M)
    assert (c.N, c.W) == (300, 100)
    rng = np.random.default_rng(0)
    U = 5e-9 * rng.standard_normal(c.W)
    for th in wlm.draw_params(wl, 5, seed=3):
        bad, zs, vs = orc.integrate(M, th, wl["z0"], wl["v0"])
        assert bad == 0
        want = 0.0
        for j in range(c.W):
            n = c.N - c.W + 1 + j
            want += (zs[n] - U[j]) ** 2
        assert orc.misfit(M, th, wl["z0"], wl["v0"], U) == pytest.approx(want, rel=1e-13, abs=0.0)
        bad, w = orc.window(M, th, wl["z0"], wl["v0"])
        assert np.array_equal(w, zs[c.N - c.W + 1:])
        # a one-sample shift of the trace is a different number (catches off-by-one)
        assert orc.misfit(M, th, wl["z0"], wl["v0"], np.roll(U, 1)) != pytest.approx(want, rel=1e-6, abs=0.0)


def test_forward_batch_segments_and_initial_states():
    wl = wlm.scaled(wlm.config(2), n_cycles=4, n_skip_cycles=2, steps_per_cycle=64)
    M = orc.model_from(wl)
    c = orc.constants(M)
    rng = np.random.default_rng(1)
    P, T = 12, 3
    params = wlm.draw_params(wl, P, seed=4)
    traces = 3e-9 * rng.standard_normal((T, c.W))
    z0v0 = wlm.draw_initial_states(wl, P, seed=5)
    got = orc.forward_batch(M, params, traces, z0v0=z0v0, n_traces=T)
    got_omp = orc.forward_batch(M, params, traces, z0v0=z0v0, n_traces=T, openmp=True)
    for p in range(P):
        want = orc.misfit(M, params[p], z0v0[p, 0], z0v0[p, 1], traces[p // (P // T)])
        assert got[p] == want
    assert np.array_equal(got, got_omp)            # the OpenMP build is the same arithmetic
    got_def = orc.forward_batch(M, params, traces, z0=wl["z0"], v0=wl["v0"], n_traces=T)
    assert got_def[0] == orc.misfit(M, params[0], wl["z0"], wl["v0"], traces[0])


def test_divergence_gives_infinity():
    wl = wlm.scaled(wlm.config(0), n_cycles=2, n_skip_cycles=1)
    M = orc.model_from(wl)
    U = np.zeros(orc.constants(M).W)
    # start beyond the |z| <= 100 A0 bound
    assert orc.misfit(M, wl["truth"], 150 * M.A0, 0.0, U) == math.inf
    # an absurdly stiff sample makes fixed-step RK4 blow up
    assert orc.misfit(M, [1e-19, 1e16], wl["z0"], wl["v0"], U) == math.inf
    bad, zs, vs = orc.integrate(M, [1e-19, 1e16], wl["z0"], wl["v0"])
    assert bad == 1 and np.isnan(zs[-1]) and np.isfinite(zs[0])
    # a sane particle is finite
    assert math.isfinite(orc.misfit(M, wl["truth"], wl["z0"], wl["v0"], U))

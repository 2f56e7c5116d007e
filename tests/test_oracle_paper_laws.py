"""Pins for the oracle's two PAPER laws (R19/R20):
Hooke, Eq. 11, and Kelvin-Voigt, Eq. 12, active
only while the tip is pressed into the sample.

Pins: hand values; reduction to the linear oscillator's closed form when the
sample is never touched or has k_s = 0; the exact piecewise-LINEAR solution
(inside the sample the cantilever is a linear oscillator with stiffness
k + k_s and damping c + zeta_s about a shifted rest position -- its closed
form is typed here independently); scipy DOP853; energy balance per cycle."""
import cmath
import math

import numpy as np
import pytest
from scipy.integrate import solve_ivp

from oracle import binding as orc
from paper_1109_0334_b200 import workloads as wlm


def _model(law, z_c=8e-9):
    return orc.Model(k=2.0, f0=70e3, Q=100.0, f_drive=70e3, A0=10e-9, z_c=z_c, R=10e-9,
                     a0=0.3e-9, law=law, n_theta=2, S=100, n_cycles=1, n_skip=0, pad_=0)


def test_hand_values():
    # Hooke, k_s = 4 N/m, h = 50 nm (the paper's truth): tip at z = -52 nm is 2 nm in
    M = _model(orc.LAW_HOOKE, z_c=8e-9)
    z = -52e-9
    assert orc.force(M, [4.0, 50e-9], z + M.z_c, 0.3) == pytest.approx(8e-9, rel=1e-13)
    assert orc.force(M, [4.0, 50e-9], -49e-9 + M.z_c, 0.3) == 0.0          # above the sample
    assert orc.force(M, [4.0, 50e-9], -50e-9 + M.z_c, 0.0) == 0.0          # continuous at touch
    # the config's z_c plays no role for Hooke: only z + h does
    M2 = _model(orc.LAW_HOOKE, z_c=3e-9)
    assert orc.force(M2, [4.0, 50e-9], z + M2.z_c, 0.0) == pytest.approx(8e-9, rel=1e-13)
    # Kelvin-Voigt, k_s = 4, zeta_s = 0.1 N s/m (the paper's truth), gap -2 nm, v = -1e-6 m/s:
    # 8e-9 + 1e-7
    K = _model(orc.LAW_KELVIN_VOIGT)
    assert orc.force(K, [4.0, 0.1], -2e-9, -1e-6) == pytest.approx(1.08e-7, rel=1e-13)
    assert orc.force(K, [4.0, 0.1], +1e-12, -1e-6) == 0.0
    # the damper acts at touch already: jump of -zeta v at gap -> 0-
    assert orc.force(K, [4.0, 0.1], -1e-30, 2e-6) == pytest.approx(-2e-7, rel=1e-9)


def _closed_form_linear(k, cdamp, m, F0, w, z0, v0, t, shift=0.0):
    """z(t) of m z'' + cdamp z' + k (z - shift) = F0 cos(w t), exact."""
    G = F0 / complex(k - m * w * w, cdamp * w)          # particular: Re(G e^{iwt})
    lam = complex(-cdamp / (2 * m), math.sqrt(k / m - (cdamp / (2 * m)) ** 2))
    a0 = z0 - shift - G.real
    b0 = v0 - (1j * w * G).real
    # homogeneous part Re(C e^{lam t}) with Re(C) = a0, Re(lam C) = b0
    Ci = (lam.real * a0 - b0) / lam.imag
    C = complex(a0, Ci)
    return shift + (G * cmath.exp(1j * w * t)).real + (C * cmath.exp(lam * t)).real


@pytest.mark.parametrize("law,theta", [(orc.LAW_HOOKE, [4.0, 50e-9]),
                                       (orc.LAW_HOOKE, [0.0, 5e-9]),
                                       (orc.LAW_KELVIN_VOIGT, [0.0, 0.0])])
def test_reduces_to_the_free_oscillator(law, theta):
    """Sample out of reach (h = 50 nm > A0) or with no stiffness and damping:
    the trajectory is the linear oscillator's closed form."""
    wl = dict(wlm.paper_law("hooke"), law=law)
    M = orc.model_from(wl, n_cycles=5, S=512, n_skip=0)
    c = orc.constants(M)
    z0, v0 = 3e-9, -1e-3
    bad, zs, vs = orc.integrate(M, theta, z0, v0)
    t = np.arange(c.N + 1) * c.dt
    ref = np.array([_closed_form_linear(M.k, c.c, c.m, c.F0, c.w, z0, v0, x) for x in t])
    assert bad == 0
    assert np.max(np.abs(zs - ref)) < 1e-6 * M.A0     # RK4 truncation at S = 512


@pytest.mark.parametrize("name", ["hooke", "kelvin_voigt"])
def test_inside_the_sample_the_solution_is_the_stiffer_linear_oscillator(name):
    """Start pressed in, moving down, and follow the closed form of the
    oscillator with k + k_s, c + zeta_s and rest position shifted by
    -k_s h/(k + k_s) until the tip leaves the sample."""
    wl = wlm.paper_law(name)
    th = wl["truth"]
    k_s = th[0]
    h = th[1] if name == "hooke" else wl["cantilever"]["z_c"]
    zeta = th[1] if name == "kelvin_voigt" else 0.0
    M = orc.model_from(wl, n_cycles=1, S=4096, n_skip=0)
    c = orc.constants(M)
    z0, v0 = -h - 0.2e-9, -2e-4
    bad, zs, vs = orc.integrate(M, th, z0, v0)
    gap = zs + h
    n_in = int(np.argmax(gap >= 0.0))          # first step outside
    assert n_in > 100
    t = np.arange(n_in) * c.dt
    ke = M.k + k_s
    ref = np.array([_closed_form_linear(ke, c.c + zeta, c.m, c.F0, c.w, z0, v0, x,
                                        shift=-k_s * h / ke) for x in t])
    assert np.max(np.abs(zs[:n_in] - ref)) < 1e-9 * M.A0


@pytest.mark.parametrize("name", ["hooke", "kelvin_voigt"])
def test_agrees_with_scipy_dop853(name):
    wl = wlm.paper_law(name)
    th, cl = wl["truth"], wl["cantilever"]
    w0, w = 2 * math.pi * cl["f0"], 2 * math.pi * cl["f_drive"]
    m = cl["k"] / w0 ** 2
    F0 = cl["k"] * cl["A0"] * math.hypot(1 - (w / w0) ** 2, (w / w0) / cl["Q"])
    h = th[1] if name == "hooke" else cl["z_c"]
    zeta = th[1] if name == "kelvin_voigt" else 0.0

    def f(t, y):
        z, v = y
        g = z + h
        fts = (-th[0] * g - zeta * v) if g < 0 else 0.0
        return [v, (F0 * math.cos(w * t) - m * w0 / cl["Q"] * v - cl["k"] * z + fts) / m]
    ncyc = 3
    T = ncyc / cl["f_drive"]
    sol = solve_ivp(f, (0.0, T), [wl["z0"], wl["v0"]], method="DOP853", rtol=1e-12,
                    atol=[1e-22, 1e-16], dense_output=True, max_step=T / (ncyc * 256))
    errs = []
    for S in (128, 256, 1024):
        M = orc.model_from(wl, n_cycles=ncyc, S=S, n_skip=0)
        c = orc.constants(M)
        bad, zs, vs = orc.integrate(M, th, wl["z0"], wl["v0"])
        assert bad == 0
        errs.append(np.max(np.abs(zs - sol.sol(np.arange(c.N + 1) * c.dt)[0])))
    # the force has a kink (Hooke) or a jump of -zeta v (Kelvin-Voigt) at touch: RK4
    # loses its order there (first order across a jump), but the error shrinks with
    # the step and is small at S = 256
    assert errs[1] < (2e-4 if name == "hooke" else 5e-3) * cl["A0"], errs
    assert errs[2] < errs[1] < errs[0], errs


def _last_cycle(wl, theta, n_cycles, S):
    M = orc.model_from(wl, n_cycles=n_cycles, S=S, n_skip=0)
    c = orc.constants(M)
    bad, zs, vs = orc.integrate(M, theta, wl["z0"], wl["v0"])
    assert bad == 0
    n = np.arange(c.N - S + 1, c.N + 1)
    drive = c.F0 * np.cos(2 * math.pi * n / S)
    return M, c, zs[-S:], vs[-S:], np.sum(drive * vs[-S:]) * c.dt, np.sum(c.c * vs[-S:] ** 2) * c.dt


def test_energy_balance_hooke_is_conservative_and_kelvin_voigt_dissipates():
    wl = wlm.paper_law("hooke")
    M, c, z, v, E_in, E_damp = _last_cycle(wl, wl["truth"], 500, 1024)
    assert z.min() + wl["truth"][1] < -0.2e-9            # the tip really presses in
    assert E_in == pytest.approx(E_damp, rel=3e-4)
    wk = wlm.paper_law("kelvin_voigt")
    th = wk["truth"]
    M, c, z, v, E_in, E_damp = _last_cycle(wk, th, 500, 2048)
    inside = (z + wk["cantilever"]["z_c"]) < 0
    E_kv = np.sum(th[1] * v[inside] ** 2) * c.dt
    assert E_kv > 0.02 * E_damp
    assert E_in - E_damp == pytest.approx(E_kv, rel=2e-2)


def test_both_unknowns_are_observable_and_truth_is_recovered_noise_free():
    """Small swarm on a noise-free trace: PSO finds the truth of each law (the
    Kelvin-Voigt landscape is corrugated: a larger swarm)."""
    for name, n_p, n_it in (("hooke", 48, 60), ("kelvin_voigt", 128, 100)):
        wl = wlm.scaled(wlm.paper_law(name), n_cycles=30, n_skip_cycles=15,
                        n_particles=n_p, n_iters=n_it)
        M = orc.model_from(wl)
        bad, win = orc.window(M, wl["truth"], wl["z0"], wl["v0"])
        o = orc.pso_invert(M, orc.box_from(wl), orc.swarm_from(wl), 0, win[None, :],
                           wl["z0"], wl["v0"])
        rel = np.abs(o["theta_star"][0] - np.array(wl["truth"])) / np.array(wl["truth"])
        assert rel.max() < 2e-2, (name, rel, o["J_star"])

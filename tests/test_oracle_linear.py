"""Pins for the oracle's integrator on the linear oscillator (F_ts = 0).

What fixes the answers here is outside the oracle: the RK4 stability
polynomial, the textbook closed form of the driven damped oscillator
(Meirovitch, ref [21] of the paper), and 4th-order convergence
("explicit 4th order Runge-Kutta").
"""
import math

import numpy as np
import pytest

from oracle import binding as orc


def _model(S=256, n_cycles=5, n_skip=0, r=1.0, Q=100.0, A0=10e-9, law=orc.LAW_NONE,
           k=2.0, f0=70e3):
    return orc.Model(k=k, f0=f0, Q=Q, f_drive=r * f0, A0=A0, z_c=8e-9, R=10e-9,
                     a0=0.3e-9, law=law, n_theta=2, S=S, n_cycles=n_cycles,
                     n_skip=n_skip, pad_=0)


def test_constants_match_definitions():
    M = _model(r=0.97, Q=37.0)
    c = orc.constants(M)
    assert c.w0 == pytest.approx(2 * math.pi * 70e3, rel=1e-15, abs=0.0)
    assert c.w == pytest.approx(2 * math.pi * 0.97 * 70e3, rel=1e-15, abs=0.0)
    assert c.m * c.w0 ** 2 == pytest.approx(M.k, rel=1e-14, abs=0.0)      # k = m w0^2
    assert c.c == pytest.approx(c.m * c.w0 / M.Q, rel=1e-14, abs=0.0)    # damping m w0/Q
    assert c.dt * M.S * M.f_drive == pytest.approx(1.0, rel=1e-14, abs=0.0)  # S steps per drive period
    assert c.N == M.S * M.n_cycles and c.W == M.S * (M.n_cycles - M.n_skip)
    # drive at resonance: F0 = k A0 / Q
    c1 = orc.constants(_model(r=1.0, Q=100.0))
    assert c1.F0 == pytest.approx(2.0 * 10e-9 / 100.0, rel=1e-14, abs=0.0)


def test_rk4_tableau_is_the_degree4_taylor_polynomial():
    """Undriven linear system x' = A x: one classical RK4 step multiplies x by
    R(hA) = I + hA + (hA)^2/2 + (hA)^3/6 + (hA)^4/24, so N steps = R^N x0.
    A wrong weight or stage coefficient changes R."""
    M = _model(S=64, n_cycles=7, A0=0.0, Q=12.0)   # A0 = 0  =>  F0 = 0
    c = orc.constants(M)
    assert c.F0 == 0.0
    A = np.array([[0.0, 1.0], [-c.w0 ** 2, -c.w0 / M.Q]])
    hA = c.dt * A
    R = np.eye(2) + hA + hA @ hA / 2 + hA @ hA @ hA / 6 + hA @ hA @ hA @ hA / 24
    x0 = np.array([3e-9, -1.1e-3])
    # A0 = 0 makes the divergence bound 100*A0 = 0, so step by hand through the public step
    z, v = x0
    x = x0.copy()
    for n in range(int(c.N)):
        z, v = orc.rk4_step(M, [0, 0], n * c.dt, c.dt, z, v)
        x = R @ x
        assert z == pytest.approx(x[0], rel=1e-11, abs=1e-24)
        assert v == pytest.approx(x[1], rel=1e-11, abs=1e-18)


def _closed_form(M, z0, v0, t):
    """Driven damped oscillator, textbook solution:
    z = A cos(w t - phi) + exp(-g t) (C1 cos(wd t) + C2 sin(wd t))."""
    w0 = 2 * math.pi * M.f0
    w = 2 * math.pi * M.f_drive
    r = w / w0
    g = w0 / (2 * M.Q)
    wd = w0 * math.sqrt(1 - 1 / (4 * M.Q ** 2))
    F0_over_k = M.A0 * math.sqrt((1 - r * r) ** 2 + (r / M.Q) ** 2)
    A = F0_over_k / math.sqrt((1 - r * r) ** 2 + (r / M.Q) ** 2)
    phi = math.atan2(r / M.Q, 1 - r * r)
    C1 = z0 - A * math.cos(phi)
    C2 = (v0 - A * w * math.sin(phi) + g * C1) / wd
    zs = A * np.cos(w * t - phi) + np.exp(-g * t) * (C1 * np.cos(wd * t) + C2 * np.sin(wd * t))
    return zs, A, phi


@pytest.mark.parametrize("r", [0.99, 1.0, 1.02])
def test_driven_linear_closed_form_and_fourth_order(r):
    """Full transient against the closed form; the error falls 16x per step
    halving (a wrong stage time c_i = (0, 1/2, 1/2, 1) would drop the order)."""
    errs = []
    for S in (50, 100, 200, 400):
        M = _model(S=S, n_cycles=5, r=r, Q=20.0)
        c = orc.constants(M)
        bad, zs, vs = orc.integrate(M, [0, 0], 4e-9, 2e-3)
        assert bad == 0
        t = np.arange(c.N + 1) * c.dt
        ref, _, _ = _closed_form(M, 4e-9, 2e-3, t)
        errs.append(np.max(np.abs(zs - ref)))
    assert errs[0] < 2e-3 * 10e-9
    ratios = [errs[i] / errs[i + 1] for i in range(3)]
    for q in ratios:
        assert 14.5 < q < 17.5, ratios


def test_steady_state_amplitude_and_phase():
    """After many decay times the response is A0 cos(w t - phi) with
    tan(phi) = (r/Q)/(1-r^2): the F0 definition makes the free amplitude A0."""
    r = 0.99
    M = _model(S=256, n_cycles=300, r=r, Q=50.0)
    c = orc.constants(M)
    bad, zs, vs = orc.integrate(M, [0, 0], 0.0, 0.0)
    assert bad == 0
    S = M.S
    last = zs[-S:]                         # samples n = N-S+1 .. N
    n = np.arange(c.N - S + 1, c.N + 1)
    ph = 2 * math.pi * n / S               # w t_n
    a = 2 / S * np.sum(last * np.cos(ph))
    b = 2 / S * np.sum(last * np.sin(ph))
    amp = math.hypot(a, b)
    phi = math.atan2(b, a)
    assert amp == pytest.approx(M.A0, rel=2e-6, abs=0.0)
    assert phi == pytest.approx(math.atan2(r / M.Q, 1 - r * r), abs=2e-6)


def test_free_steady_state_initial_condition_stays_on_orbit():
    """Starting ON the free orbit (the workloads' default z0, v0) the F_ts = 0
    trajectory is A0 sin(w t) at resonance from step 0."""
    from paper_1109_0334_b200 import workloads as wlm
    wl = wlm.config(1)
    M = orc.model_from(wl, law=orc.LAW_NONE, n_cycles=3)
    c = orc.constants(M)
    bad, zs, vs = orc.integrate(M, [0, 0], wl["z0"], wl["v0"])
    t = np.arange(c.N + 1) * c.dt
    assert np.max(np.abs(zs - M.A0 * np.sin(c.w * t))) < 1e-6 * M.A0


def test_time_is_not_accumulated():
    """t_n = n*dt: integrating 2N steps equals integrating N steps and then
    N more started at step index N only if the drive phase is taken from n*dt;
    check the drive phase after many cycles against cos(2 pi n / S)."""
    M = _model(S=128, n_cycles=1)
    c = orc.constants(M)
    n = 128 * 5000 + 17
    dz, dv = orc.rhs(M, [0, 0], n * c.dt, 0.0, 0.0)
    assert dv * c.m == pytest.approx(c.F0 * math.cos(2 * math.pi * 17 / 128), rel=1e-9, abs=0.0)

"""Pins for the oracle's multi-mode Euler-Bernoulli forward model (the paper's own
forward problem, Appendix A/B).

What fixes it from outside the oracle: the numbers the paper prints in Appendix A
(first natural frequency 25 468.9 Hz; steady-state deflection amplitude 3.2 um
for a 5 nm base motion at 25 500 Hz), the textbook roots and boundary conditions
of the clamped-free beam, orthogonality of the modes, the closed-form response
of each (linear) modal oscillator, the already-pinned point-mass oracle in the
one-mode case, and an independent library integrator (scipy DOP853) on the
16-dimensional system typed here in numpy with modal constants computed here."""
import cmath
import math

import numpy as np
import pytest
from scipy.integrate import solve_ivp
from scipy.optimize import brentq

from oracle import binding as orc
from paper_1109_0334_b200 import workloads as wlm

ROOTS = [1.875104068711961, 4.694091132974175, 7.854757438237613, 10.995540734875467]


@pytest.fixture(scope="module")
def setup():
    wl = wlm.beam_workload()
    B = orc.beam_from(wl)
    return wl, B, orc.beam_setup(B)


def test_appendix_a_first_natural_frequency_and_textbook_roots(setup):
    wl, B, mo = setup
    # PAPER.md:311 "First natural frequency | 25468.9 Hz"
    assert mo.omega[0] / (2 * math.pi) == pytest.approx(25468.9, abs=0.05)
    for i, r in enumerate(ROOTS):
        assert mo.bL[i] == pytest.approx(r, rel=1e-13)
    for i in range(4, 8):                      # asymptotically (i + 1/2) pi
        assert mo.bL[i] == pytest.approx((i + 0.5) * math.pi, abs=1e-5)
        assert abs(math.cos(mo.bL[i]) * math.cosh(mo.bL[i]) + 1) < 1e-4 * math.cosh(mo.bL[i])
    assert mo.omega[1] / mo.omega[0] == pytest.approx(6.2669, rel=1e-4)    # textbook ratios
    assert mo.omega[2] / mo.omega[0] == pytest.approx(17.5475, rel=1e-4)
    # PAPER.md:304 the area moment of the 35 x 5 um section
    assert B.I == pytest.approx(3.64583e-22, rel=1e-5)


def test_appendix_a_steady_state_amplitude_3_2_microns(setup):
    """base amplitude 5 nm at 25 500 Hz, 8 modes, no damping in
    the table: the particular solution of every modal equation summed at the tip,
    |A_b w^2 sum_i Phi_i(L) <1,Phi_i>/<Phi_i,Phi_i> / (w_i^2 - w^2)| = 3.2 um."""
    wl, B, mo = setup
    w = 2 * math.pi * 25500.0
    amp = sum(mo.phiL[i] * mo.intphi[i] / mo.norm[i] / (mo.omega[i] ** 2 - w * w)
              for i in range(8)) * 5e-9 * w * w
    assert abs(amp) == pytest.approx(3.2e-6, abs=0.05e-6)
    # and the integrator reproduces that amplitude: undamped (Q huge), from the
    # particular solution's own initial state, the tip stays on it
    Bu = orc.beam_from(wl, law=0, Q=1e12, f_drive=25500.0, A_base=5e-9, A_ref=1.0, S=1024,
                       n_cycles=3, n_skip=0)
    mu = orc.beam_setup(Bu)
    eta0 = [mu.gain[i] / (mu.omega[i] ** 2 - w * w) for i in range(8)] + [0.0] * 8
    bad, u, v, _ = orc.beam_integrate(Bu, [0, 0], eta0=eta0)
    assert bad == 0
    assert (u.max() - u.min()) / 2 == pytest.approx(abs(amp), rel=1e-6)


def _phi_textbook(bL, xi):
    s = (math.cosh(bL) + math.cos(bL)) / (math.sinh(bL) + math.sin(bL))
    return (math.cosh(bL * xi) - math.cos(bL * xi)) - s * (math.sinh(bL * xi) - math.sin(bL * xi))


def test_mode_shapes_eq6_boundary_conditions_orthogonality_and_eq7_reading(setup):
    wl, B, mo = setup
    L = B.L
    xs = np.linspace(0.0, L, 4001)
    Phi = np.array([[orc.beam_shape(B, mo, i, x) for x in xs] for i in range(8)])
    h = xs[1] - xs[0]
    for i in range(8):
        p = Phi[i]
        scale = np.abs(p).max()
        b = mo.bL[i] / L
        assert abs(p[0]) < 1e-12 * scale                                    # Phi(0) = 0
        assert abs((p[1] - p[0]) / h) < 2e-3 * scale * b * (1 + b * h * 200)  # Phi'(0) = 0
        d2 = (p[-1] - 2 * p[-2] + p[-3]) / h ** 2                           # Phi''(L) = 0
        assert abs(d2) < 2e-2 * scale * b * b
        d3 = (p[-1] - 3 * p[-2] + 3 * p[-3] - p[-4]) / h ** 3               # Phi'''(L) = 0
        assert abs(d3) < 5e-2 * scale * b ** 3
    # Eq. 6 equals the textbook hyperbolic form up to a constant factor (low modes)
    for i in range(3):
        ref = np.array([_phi_textbook(mo.bL[i], x / L) for x in xs])
        ratio = Phi[i][1:] / ref[1:]
        assert np.ptp(ratio[np.abs(ref[1:]) > 1e-3]) < 1e-9 * abs(ratio[-1])
    # orthogonality over the length (the Gram matrix is diagonal)
    w = np.full(xs.size, h)
    w[0] = w[-1] = h / 2
    gram = (Phi * w) @ Phi.T
    dg = np.sqrt(np.diag(gram))
    off = gram / np.outer(dg, dg) - np.eye(8)
    assert np.abs(off).max() < 1e-5
    # Simpson with the paper's 501 points against this finer quadrature
    for i in range(8):
        assert mo.norm[i] == pytest.approx(gram[i, i], rel=2e-5)
        assert mo.intphi[i] == pytest.approx(float(Phi[i] @ w), rel=1e-4, abs=1e-9 * L)
    # first-mode participation factor Phi(L) <1,Phi>/<Phi,Phi> = 1.566 (textbook)
    assert mo.phiL[0] * mo.intphi[0] / mo.norm[0] == pytest.approx(1.5660, rel=1e-4)
    # DESIGN.md R22: Eq. 7 exactly as printed does NOT satisfy the free-end condition
    Bl = orc.beam_from(wl, literal_eq7=1)
    ml = orc.beam_setup(Bl)
    p = np.array([orc.beam_shape(Bl, ml, 0, x) for x in xs])
    d2 = (p[-1] - 2 * p[-2] + p[-3]) / h ** 2
    assert abs(d2) > 0.02 * np.abs(p).max() * (mo.bL[0] / L) ** 2


def _modal_closed_form(w_i, Q, g, w, t):
    """eta(t) of eta'' + (w_i/Q) eta' + w_i^2 eta = g cos(w t) from rest."""
    c = w_i / Q
    G = g / complex(w_i ** 2 - w * w, c * w)
    lam = complex(-c / 2, math.sqrt(w_i ** 2 - c * c / 4))
    a0 = -G.real
    b0 = -(1j * w * G).real
    C = complex(a0, (lam.real * a0 - b0) / lam.imag)
    return (G * cmath.exp(1j * w * t)).real + (C * cmath.exp(lam * t)).real


def _linear_tip_error(wl, n_modes, S, n_cycles=6):
    Bn = orc.beam_from(wl, law=0, S=S, n_cycles=n_cycles, n_skip=0, n_modes=n_modes)
    mn = orc.beam_setup(Bn)
    bad, u, v, eta = orc.beam_integrate(Bn, [0, 0], want_eta=True)
    assert bad == 0
    t = np.arange(mn.N + 1) * mn.dt
    ref = np.zeros_like(t)
    per_mode = []
    for i in range(n_modes):
        e_i = np.array([_modal_closed_form(mn.omega[i], Bn.Q, mn.gain[i], mn.w, x) for x in t])
        ref += mn.phiL[i] * e_i
        per_mode.append(np.max(np.abs(eta[:, i] - e_i)) * abs(mn.phiL[i]))
    return np.max(np.abs(u - ref)), per_mode, np.max(np.abs(ref))


def test_linear_response_is_the_sum_of_modal_closed_forms_and_fourth_order(setup):
    wl, B, mo = setup
    # all 8 modes at the workload's own step: every mode's contribution to the tip
    # follows its closed form (the stiff modes' short transients are where RK4 at
    # h w_8 = 1.94 is least accurate; they carry 1e-4 of the deflection)
    err, per_mode, scale = _linear_tip_error(wl, 8, 512)
    assert err < 2e-5 * scale
    assert max(per_mode) < 2e-5 * scale and per_mode[0] < 1e-8 * scale
    # order of convergence on the three lowest modes (h w_3 = 0.2 at S = 512)
    errs = [_linear_tip_error(wl, 3, S)[0] for S in (256, 512, 1024)]
    assert 13 < errs[0] / errs[1] < 19 and 13 < errs[1] / errs[2] < 19, errs


def test_one_mode_beam_is_the_point_mass_oracle(setup):
    """m = 1: u = Phi(L) eta obeys m_eff u'' + (m_eff w1/Q) u' + k_eff u =
    F0 cos(w t) + F_ts(u + z_c), m_eff = mu <Phi,Phi>/Phi(L)^2 -- exactly the
    point-mass model of afm_oracle.c, whose pins then carry over."""
    wl, B, mo = setup
    B1 = orc.beam_from(wl, n_modes=1, n_cycles=30, n_skip=15)
    m1 = orc.beam_setup(B1)
    m_eff = 1.0 / (m1.phiL[0] * m1.fgain[0])
    k_eff = m_eff * m1.omega[0] ** 2
    F0 = m_eff * m1.phiL[0] * m1.gain[0]
    r = m1.w / m1.omega[0]
    A0 = F0 / (k_eff * math.hypot(1 - r * r, r / B1.Q))
    M = orc.Model(k=k_eff, f0=m1.omega[0] / (2 * math.pi), Q=B1.Q, f_drive=B1.f_drive, A0=A0,
                  z_c=B1.z_c, R=B1.R, a0=B1.a0, law=B1.law, n_theta=2, S=B1.S,
                  n_cycles=B1.n_cycles, n_skip=B1.n_skip, pad_=0)
    assert k_eff == pytest.approx(3 * B1.E * B1.I / B1.L ** 3, rel=0.04)   # ~ static 3EI/L^3
    bad1, u, v, _ = orc.beam_integrate(B1, wl["truth"])
    bad2, zs, vs = orc.integrate(M, wl["truth"], 0.0, 0.0)
    assert bad1 == 0 and bad2 == 0
    assert u.min() + B1.z_c < B1.a0                  # the tip reaches contact
    assert np.max(np.abs(u - zs)) < 1e-9 * np.max(np.abs(zs))


def test_nonlinear_eight_mode_solution_against_scipy_dop853(setup):
    """The 16-dimensional system typed independently: roots by brentq, shapes
    by the textbook formula, inner products by a fine trapezoid rule, DMT force
    in numpy; DOP853 at rtol 1e-11.  RK4 at S = 512 .. 2048 converges to it."""
    wl, B, mo = setup
    m, L = 8, B.L
    bL = [brentq(lambda x: math.cos(x) + 1 / math.cosh(x), (i + 0.5) * math.pi - 0.4,
                 (i + 0.5) * math.pi + 0.4, xtol=1e-15) for i in range(m)]
    xi = np.linspace(0, 1, 20001)

    def shape(i):
        # exponential-safe evaluation of the textbook form
        b = bL[i]
        s = (1 + math.exp(-2 * b) + 2 * math.exp(-b) * math.cos(b)) / \
            (1 - math.exp(-2 * b) + 2 * math.exp(-b) * math.sin(b))
        return (0.5 * ((1 - s) * np.exp(b * (xi - 1)) * math.exp(b) if b < 30 else 0) +
                0.5 * (1 + s) * np.exp(-b * xi) - np.cos(b * xi) + s * np.sin(b * xi))
    ph = [shape(i) for i in range(m)]
    wq = np.full(xi.size, L / (xi.size - 1))
    wq[0] = wq[-1] = wq[0] / 2
    N = [float((p * p) @ wq) for p in ph]
    Ip = [float(p @ wq) for p in ph]
    pL = [float(p[-1]) for p in ph]
    om = [b * b * math.sqrt(B.E * B.I / (B.mu * L ** 4)) for b in bL]
    w = 2 * math.pi * B.f_drive
    gain = [B.A_base * w * w * Ip[i] / N[i] for i in range(m)]
    fg = [pL[i] / (B.mu * N[i]) for i in range(m)]
    H, Es = wl["truth"]

    def rhs(t, y):
        u = sum(pL[i] * y[i] for i in range(m))
        d = u + B.z_c
        if d > B.a0:
            F = -H * B.R / (6 * d * d)
        else:
            F = -H * B.R / (6 * B.a0 ** 2) + 4 / 3 * Es * math.sqrt(B.R) * (B.a0 - d) ** 1.5
        return list(y[m:]) + [gain[i] * math.cos(w * t) - om[i] / B.Q * y[m + i]
                              - om[i] ** 2 * y[i] + fg[i] * F for i in range(m)]
    ncyc = 40                                   # contact starts near cycle 26
    T = ncyc / B.f_drive
    sol = solve_ivp(rhs, (0, T), [0.0] * 16, method="DOP853", rtol=1e-11, atol=1e-24,
                    dense_output=True, max_step=T / (ncyc * 128))
    errs = []
    for S in (512, 2048):
        Bs = orc.beam_from(wl, S=S, n_cycles=ncyc, n_skip=0)
        ms = orc.beam_setup(Bs)
        bad, u, v, _ = orc.beam_integrate(Bs, wl["truth"])
        assert bad == 0
        t = np.arange(ms.N + 1) * ms.dt
        y = sol.sol(t)
        ref = sum(pL[i] * y[i] for i in range(m))
        errs.append(np.max(np.abs(u - ref)))
    assert u.min() + B.z_c < B.a0               # contact happened within these cycles
    assert errs[0] < 2e-3 * B.A_ref and errs[1] < errs[0], errs


def test_misfit_window_batch_and_inversion_wiring(setup):
    wl, B, mo = setup
    Bs = orc.beam_from(wl, n_cycles=30, n_skip=15)
    ms = orc.beam_setup(Bs)
    bad, win = orc.beam_window(Bs, wl["truth"])
    bad2, u, _, _ = orc.beam_integrate(Bs, wl["truth"])
    assert bad == 0 and np.array_equal(win, u[-ms.W:])
    rng = np.random.default_rng(1)
    noise = 1e-11 * rng.standard_normal(ms.W)
    params = np.array([wl["truth"], [3e-19, 2e9]])
    J = orc.beam_forward_batch(Bs, params, win + noise)
    assert J[0] == pytest.approx(float(noise @ noise), rel=1e-9)
    bad3, u3, _, _ = orc.beam_integrate(Bs, params[1])
    assert J[1] == pytest.approx(float(np.sum((u3[-ms.W:] - win - noise) ** 2)), rel=1e-12)
    assert J[1] > 100 * J[0]
    # diverging trajectory -> +Inf (tiny reference amplitude)
    Bd = orc.beam_from(wl, n_cycles=30, n_skip=15, A_ref=1e-11)
    assert np.isinf(orc.beam_forward_batch(Bd, params[:1], win)[0])
    # the PSO loop is the pinned one of afm_oracle.c: same streams, same rules
    w2 = wlm.scaled(wl, n_cycles=30, n_skip_cycles=15, n_particles=6, n_iters=3)
    o = orc.beam_pso_invert(Bs, orc.box_from(w2), orc.swarm_from(w2), 0, win, dump=True)
    a, b = orc.pso_uniforms(0, 4, 0, 0, 2)
    lo, hi = np.array(wl["bounds"]["lo"]), np.array(wl["bounds"]["hi"])
    assert np.array_equal(o["dump"][0, 4, 0:2], lo + a * (hi - lo))
    th = wlm.theta_of_coords(wl, o["dump"][1, :, 0:2])
    assert np.array_equal(o["dump"][1, :, 6], orc.beam_forward_batch(Bs, th, win))
    assert o["J_star"][0] == o["dump"][:, :, 6].min()

"""Pins for the oracle's tip-sample force laws and right-hand side
(BASELINE.json configs[0], [2], [3]; named at PAPER.md:78)."""
import math
import os

import numpy as np
import pytest

from oracle import binding as orc

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "force_hand_values.txt")


def _model(law, R=10e-9, a0=0.3e-9, z_c=8e-9):
    return orc.Model(k=2.0, f0=70e3, Q=100.0, f_drive=70e3, A0=10e-9, z_c=z_c, R=R,
                     a0=a0, law=law, n_theta=4, S=100, n_cycles=1, n_skip=0, pad_=0)


def test_hand_values_from_golden_file():
    laws = {"DMT": orc.LAW_DMT, "DMT_VISC": orc.LAW_DMT_VISC}
    n = 0
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        law, H, Es, eta, R, a0, d, v, F = line.split()
        M = _model(laws[law], R=float(R), a0=float(a0))
        got = orc.force(M, [float(H), float(Es), float(eta), 0.0], float(d), float(v))
        assert got == pytest.approx(float(F), rel=1e-13, abs=0.0), line
        n += 1
    assert n == 5


def test_dmt_is_continuous_at_a0_and_repulsive_deep_in_contact():
    M = _model(orc.LAW_DMT)
    th = [1e-19, 1e9]
    a0 = M.a0
    below = orc.force(M, th, a0 * (1 - 1e-12))
    at = orc.force(M, th, a0)
    above = orc.force(M, th, a0 * (1 + 1e-12))
    assert below == pytest.approx(at, rel=1e-9, abs=0.0)
    assert above == pytest.approx(at, rel=1e-9, abs=0.0)
    assert at < 0                                 # adhesive plateau
    assert orc.force(M, th, a0 - 2e-9) > 0        # Hertz repulsion wins
    # attraction decays as 1/d^2
    assert orc.force(M, th, 2e-9) / orc.force(M, th, 4e-9) == pytest.approx(4.0, rel=1e-14, abs=0.0)
    # d <= 0 (deep indentation) is legal
    assert math.isfinite(orc.force(M, th, -3e-9))


def test_hertz_three_halves_power():
    M = _model(orc.LAW_DMT)
    th = [0.0, 3e9]          # H = 0 isolates the Hertz term
    f1 = orc.force(M, th, M.a0 - 1e-9)
    f4 = orc.force(M, th, M.a0 - 4e-9)
    assert f4 / f1 == pytest.approx(8.0, rel=1e-14, abs=0.0)      # 4^{3/2}
    assert f1 == pytest.approx((4 / 3) * 3e9 * 1e-4 * 1e-9 ** 1.5, rel=1e-13, abs=0.0)


def test_viscous_term_only_in_contact_vanishes_at_a0_and_opposes_motion():
    M = _model(orc.LAW_DMT_VISC)
    th = [1e-19, 1e9, 250.0]
    # out of contact: velocity has no effect
    assert orc.force(M, th, 1e-9, 0.3) == orc.force(M, th, 1e-9, -0.3)
    # at d = a0 the sqrt(R delta) factor is zero
    assert orc.force(M, th, M.a0, 0.3) == orc.force(M, th, M.a0, 0.0)
    d = M.a0 - 0.5e-9
    f0 = orc.force(M, th, d, 0.0)
    fp = orc.force(M, th, d, +1e-3)
    fm = orc.force(M, th, d, -1e-3)
    assert fp < f0 < fm
    assert f0 - fp == pytest.approx(250.0 * math.sqrt(10e-9 * 0.5e-9) * 1e-3, rel=1e-9, abs=0.0)
    # DMT law ignores the third parameter
    Md = _model(orc.LAW_DMT)
    assert orc.force(Md, th, d, 1e-3) == f0


def test_lj_exp_term_by_term_against_pow_and_exp():
    M = _model(orc.LAW_LJ_EXP)
    rng = np.random.default_rng(5)
    for _ in range(50):
        Crep, Catt, Fad, lam = 10 ** rng.uniform(-82, -80), 10 ** rng.uniform(-29, -27), \
            10 ** rng.uniform(-10, -8), 10 ** rng.uniform(-10, -8)
        d = rng.uniform(0.3e-9, 30e-9)
        want = Crep * math.pow(d, -8) - Catt * math.pow(d, -2) - Fad * math.exp(-d / lam)
        got = orc.force(M, [Crep, Catt, Fad, lam], d, rng.normal())
        assert got == pytest.approx(want, rel=1e-12, abs=1e-25)
    # each term alone, sign included
    assert orc.force(M, [1e-81, 0, 0, 1e-9], 1e-9) == pytest.approx(1e-9, rel=1e-12, abs=0.0)
    assert orc.force(M, [0, 1e-28, 0, 1e-9], 1e-9) == pytest.approx(-1e-10, rel=1e-12, abs=0.0)
    assert orc.force(M, [0, 0, 1e-9, 1e-9], 2e-9) == pytest.approx(-1e-9 * math.exp(-2), rel=1e-12, abs=0.0)


def test_rhs_by_hand():
    """a = [F0 cos(w t) - c v - k z + F_ts(z + z_c)]/m with every term typed in."""
    M = _model(orc.LAW_DMT)
    th = [1e-19, 1e9]
    w0 = 2 * math.pi * 70e3
    m = 2.0 / w0 ** 2
    F0 = 2.0 * 10e-9 / 100.0
    t, z, v = 1.3e-6, -7.2e-9, 2.5e-3
    d = z + 8e-9                                  # 0.8 nm > a0: vdW branch
    F = -1e-19 * 10e-9 / (6 * d * d)
    want = (F0 * math.cos(w0 * t) - (m * w0 / 100.0) * v - 2.0 * z + F) / m
    dz, dv = orc.rhs(M, th, t, z, v)
    assert dz == v
    assert dv == pytest.approx(want, rel=1e-12, abs=0.0)
    # the gap is z + z_c: moving the sample by dz_c is the same as moving the tip
    M2 = _model(orc.LAW_DMT, z_c=7e-9)
    assert orc.rhs(M2, th, t, z + 1e-9, v)[1] * m + 2.0 * (z + 1e-9) == \
        pytest.approx(dv * m + 2.0 * z, rel=1e-9, abs=0.0)

"""Host-side checks of constants the CUDA kernels carry (no GPU needed).

exp_fast (csrc/afm_device.cuh) evaluates exp(f), |f| <= ln2/2, by a degree-11
polynomial whose coefficients are typed into the source.  They are read back from
the source here and the polynomial is evaluated with mpmath at 50 digits: its
relative error must stay below 2e-17 on the reduced range (and a little beyond it,
since n = rint(x log2 e) comes from one fused multiply-add), and the two-part ln 2
of the range reduction must add up to ln 2.
"""
import os
import re

import pytest

mp = pytest.importorskip("mpmath")   # a box without mpmath skips this file, the rest still collects

SRC = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))),
                   "paper_1109_0334_b200", "csrc", "afm_device.cuh")


def _exp_fast_body():
    s = open(SRC).read()
    a = s.index("__device__ __forceinline__ double exp_fast(double x)")
    return s[a:s.index("\n}\n", a)]


def test_exp_fast_polynomial_is_accurate_to_2e_17():
    body = _exp_fast_body()
    pairs = re.findall(r"const double a(\d) = fma\(f, ([0-9.e+-]+), ([0-9.e+-]+)\);", body)
    assert [int(k) for k, _, _ in pairs] == [1, 2, 3, 4, 5]
    assert "const double a0 = f + 1.0;" in body
    coef = [mp.mpf(1), mp.mpf(1)]
    for _, hi, lo in pairs:          # a_k = c_{2k} + c_{2k+1} f
        coef += [mp.mpf(float(lo)), mp.mpf(float(hi))]
    assert len(coef) == 12
    mp.mp.dps = 50
    half = mp.log(2) / 2 * mp.mpf("1.002")
    worst = mp.mpf(0)
    for i in range(4001):
        f = -half + 2 * half * i / 4000
        p = sum(c * f ** k for k, c in enumerate(coef))
        worst = max(worst, abs(p / mp.exp(f) - 1))
    assert worst < mp.mpf("2e-17"), worst
    # the Taylor polynomial of the same degree is some 280 times worse
    taylor = abs(sum(half ** k / mp.factorial(k) for k in range(12)) / mp.exp(half) - 1)
    assert taylor > 100 * worst


def test_exp_fast_range_reduction_constants():
    body = _exp_fast_body()
    hi, lo = re.findall(r"fma\(n, (-[0-9.e+-]+), (?:x|f)\)", body)
    mp.mp.dps = 50
    ln2 = -(mp.mpf(float(hi)) + mp.mpf(float(lo)))
    assert abs(ln2 / mp.log(2) - 1) < mp.mpf("1e-25")
    # the high part has trailing zero bits, so n * hi is exact for |n| < 2^20
    m, _ = mp.frexp(mp.mpf(float(hi)))
    assert (m * 2 ** 33) == mp.floor(m * 2 ** 33)
    log2e = re.search(r"fma\(x, ([0-9.]+), magic\)", body).group(1)
    assert abs(mp.mpf(float(log2e)) * mp.log(2) - 1) < mp.mpf("2e-16")
    assert "max(min(__double2loint(nm), 1024), -1022)" in body

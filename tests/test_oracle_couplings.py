"""Pins T1/T2: J*(r) of Eq. 5-7 and its int32 quantisation."""
import math

import mpmath
import numpy as np
import pytest
from scipy.special import zeta as hurwitz

CASES = [(8, 0.5), (64, 0.5), (256, 0.4), (1024, 0.8), (4096, 0.3), (2048, 0.1), (2048, 1.0)]


@pytest.mark.parametrize("L,sigma", CASES)
def test_symmetry_and_positivity(oracle, L, sigma):
    J = oracle.jstar(L, sigma)
    assert J[0] == 0.0
    r = np.arange(1, L)
    assert np.all(J[1:] > 0)
    np.testing.assert_allclose(J[r], J[L - r], rtol=2e-15)
    # decreasing towards L/2
    assert np.all(np.diff(J[1 : L // 2 + 1]) < 0)


@pytest.mark.parametrize("L,sigma", [(8, 0.5), (64, 0.5), (256, 0.4)])
def test_eq5_brute_force_image_sum(oracle, L, sigma):
    """Eq. 5 written out: sum over |n| <= N of |r+nL|^-s, plus the integral of the tail
    (midpoint rule: sum_{n>N} f(n) ~ int_{N+1/2}^inf f, error O(N^-s-2))."""
    s = 1.0 + sigma
    N = 200000
    n = np.arange(1, N + 1, dtype=np.float64)
    J = oracle.jstar(L, sigma)
    for r in (1, 2, L // 4, L // 2 - 1, L // 2, L - 3):
        direct = r ** -s + np.sum((n * L + r) ** -s) + np.sum((n * L - r) ** -s)
        a = (N + 0.5) * L
        tail = ((a + r) ** (1 - s) + (a - r) ** (1 - s)) / ((s - 1) * L)
        assert J[r] == pytest.approx(direct + tail, rel=1e-11)


@pytest.mark.parametrize("L,sigma", CASES)
def test_eq6_against_library_hurwitz(oracle, L, sigma):
    """Eq. 6 with an independent Hurwitz zeta (mpmath 30 digits; scipy as a second opinion)."""
    mpmath.mp.dps = 30
    s = mpmath.mpf(1) + mpmath.mpf(sigma)     # exact sum of the two doubles, as the oracle forms it
    J = oracle.jstar(L, sigma)
    for r in sorted({1, 2, 3, L // 3, L // 2 - 1, L // 2}):
        x = mpmath.mpf(r) / L
        ref = mpmath.mpf(r) ** -s + mpmath.mpf(L) ** -s * (mpmath.zeta(s, 1 + x) + mpmath.zeta(s, 1 - x))
        assert abs(J[r] / float(ref) - 1.0) < 4e-16
        sf = float(s)
        ref2 = r ** -sf + L ** -sf * (hurwitz(sf, 1 + r / L) + hurwitz(sf, 1 - r / L))
        assert J[r] == pytest.approx(ref2, rel=1e-13)


@pytest.mark.parametrize("L", [8, 64, 2048])
def test_sigma_one_closed_form(oracle, L):
    """sigma=1: sum_n (r+nL)^-2 = (pi/L)^2 / sin^2(pi r/L)  (textbook partial-fraction series)."""
    J = oracle.jstar(L, 1.0)
    # r <= L/2 only: for r near L, fp64 sin(pi r/L) itself loses ~L eps to cancellation in the
    # argument; the upper half is pinned through the symmetry test above.
    r = np.arange(1, L // 2 + 1)
    ref = (math.pi / L) ** 2 / np.sin(math.pi * r / L) ** 2
    np.testing.assert_allclose(J[r], ref, rtol=5e-14)
    np.testing.assert_allclose(J[L - r], ref, rtol=5e-14)


@pytest.mark.parametrize("L,sigma", CASES)
def test_sum_rule(oracle, L, sigma):
    """sum_{r=1}^{L-1} J*(r) = 2 zeta(1+sigma) (1 - L^-(1+sigma)): every integer m != 0 that is not
    a multiple of L appears exactly once as r+nL."""
    s = 1.0 + sigma
    J = oracle.jstar(L, sigma)
    ref = 2.0 * float(mpmath.zeta(s)) * (1.0 - L ** -s)
    assert math.fsum(J[1:]) == pytest.approx(ref, rel=1e-13)


@pytest.mark.parametrize("L,sigma", CASES)
def test_quantiser(oracle, L, sigma):
    """A16: Jq[r] = round(J*(r) 2^24), Jq[0]=0, exact integer symmetry, no entry near a rounding tie
    (so any <=1e-12-accurate evaluation gives the same integers), row sum < 2^31."""
    J = oracle.jstar(L, sigma)
    Jq = oracle.couplings(L, sigma)
    assert Jq.dtype == np.int32 and Jq[0] == 0
    r = np.arange(1, L)
    assert np.array_equal(Jq[r], Jq[L - r])
    mpmath.mp.dps = 30
    scaled = J * 2.0 ** 24
    assert np.array_equal(Jq[1:], np.rint(scaled[1:]).astype(np.int64))
    frac = np.abs(scaled[1:] - np.floor(scaled[1:]) - 0.5)
    assert frac.min() > 1e-6
    assert int(Jq.astype(np.int64).sum()) < 2 ** 31


def test_printed_values_L8(oracle):
    """Independent 40-digit evaluation (mpmath) of Eq. 6 at L=8, sigma=0.5, quantised here."""
    mpmath.mp.dps = 40
    L, s = 8, mpmath.mpf("1.5")
    ref = [0]
    for r in range(1, L):
        x = mpmath.mpf(r) / L
        v = mpmath.mpf(r) ** -s + mpmath.mpf(L) ** -s * (mpmath.zeta(s, 1 + x) + mpmath.zeta(s, 1 - x))
        ref.append(int(mpmath.nint(v * 2 ** 24)))
    assert [int(v) for v in oracle.couplings(8, 0.5)] == ref
    # SURVEY.md 8(c) T1 lists the same integers (surveyor's scratch values)
    assert ref[1:] == [20701016, 10017126, 7631696, 7083178, 7631696, 10017126, 20701016]

"""Pins for the oracle's Wigner d-function providers (E explicit sum, R Risbo, T l-recurrence).

Everything here is checked against something other than the oracle itself: closed forms, library routines
(scipy / mpmath Jacobi polynomials, Eq. 22 of the paper), exact identities (Eq. 24, 28, 29, symmetries,
orthogonality).  SURVEY.md 8(c) pins 1-5.
"""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy.special import eval_jacobi, gammaln

LD = np.longdouble


def jacobi_d(l, m, n, beta):
    """Eq. 22-23 evaluated with scipy's Jacobi polynomial (double precision)."""
    mu, nu = abs(m - n), abs(m + n)
    s = l - (mu + nu) // 2
    zeta = 1.0 if n >= m else (-1.0) ** (n - m)
    lg = 0.5 * (gammaln(s + 1) + gammaln(s + mu + nu + 1) - gammaln(s + mu + 1) - gammaln(s + nu + 1))
    return zeta * math.exp(lg) * math.sin(beta / 2) ** mu * math.cos(beta / 2) ** nu * eval_jacobi(s, mu, nu, math.cos(beta))


def jacobi_d_mp(l, m, n, beta):
    """Eq. 22-23 at 60 digits with mpmath; returns an mpf (can be far outside double range)."""
    mu, nu = abs(m - n), abs(m + n)
    s = l - (mu + nu) // 2
    zeta = 1 if n >= m else (-1) ** (n - m)
    pre = mp.sqrt(mp.factorial(s) * mp.factorial(s + mu + nu) / (mp.factorial(s + mu) * mp.factorial(s + nu)))
    return zeta * pre * mp.sin(beta / 2) ** mu * mp.cos(beta / 2) ** nu * mp.jacobi(s, mu, nu, mp.cos(beta))


def test_eq22_normalisation_is_the_paper_convention():
    # Eq. 22's prefactor as printed is sqrt(s!(s+mu+nu)!/((s+mu)!(s-nu)!)) -- the last factor is a typo for (s+nu)!
    # (the printed form is undefined for nu > s).  d^1_{10} = -sin(b)/sqrt(2) fixes sign and normalisation.
    b = 0.7
    assert abs(jacobi_d(1, 1, 0, b) - (-math.sin(b) / math.sqrt(2))) < 1e-15
    assert abs(jacobi_d(1, 0, 1, b) - (math.sin(b) / math.sqrt(2))) < 1e-15


@pytest.mark.parametrize("beta", [0.3, 1.1, 2.9])
def test_closed_forms(orc, beta):
    b = LD(beta)
    c, s = np.cos(b), np.sin(b)
    cases = {
        (1, 0, 0): c, (1, 1, 0): -s / np.sqrt(LD(2)), (1, 1, 1): (1 + c) / 2, (1, 1, -1): (1 - c) / 2,
        (2, 0, 0): (3 * c * c - 1) / 2, (2, 2, 0): np.sqrt(LD(6)) / 4 * s * s,
        (2, 2, 2): ((1 + c) / 2) ** 2, (2, 2, -2): ((1 - c) / 2) ** 2, (2, 1, 0): -np.sqrt(LD(3) / 2) * s * c,
    }
    R = orc.d_risbo(3, b)
    for (l, m, n), want in cases.items():
        assert abs(orc.d_explicit(l, m, n, b) - want) < 1e-18
        assert abs(R[l][m + l, n + l] - want) < 1e-18
        assert abs(orc.d_lrec(3, m, n, beta=b)[l] - want) < 1e-18


def test_poles_eq28_eq29(orc):
    L = 10
    R0 = orc.d_risbo(L, LD(0))
    Rpi = orc.d_risbo(L, LD(np.pi) if False else np.arccos(LD(-1)))
    for l in range(L):
        k = 2 * l + 1
        assert np.abs(R0[l] - np.eye(k)).max() < 1e-18                      # Eq. 28: d(0) = delta_mn
        want = np.zeros((k, k), dtype=LD)
        for m in range(-l, l + 1):
            want[m + l, -m + l] = (-1.0) ** (l + m)                           # Eq. 29
        assert np.abs(Rpi[l] - want).max() < 1e-16


def test_orthogonality_and_symmetries(orc):
    L, b = 14, LD(0.83)
    R = orc.d_risbo(L, b)
    Rm = orc.d_risbo(L, np.arccos(LD(-1)) - b)
    for l in range(L):
        D = R[l]
        k = 2 * l + 1
        assert np.abs(D.T @ D - np.eye(k)).max() < 1e-17                     # sum_m d_mn d_mn' = delta
        idx = np.arange(-l, l + 1)
        sg = (-1.0) ** (idx[:, None] - idx[None, :])
        assert np.abs(D - sg * D.T).max() < 1e-17                             # d_mn = (-1)^{m-n} d_nm
        assert np.abs(D - sg * D[::-1, ::-1]).max() < 1e-17                   # = (-1)^{m-n} d_{-m,-n}
        assert np.abs(D - D[::-1, ::-1].T).max() < 1e-17                      # = d_{-n,-m}
        sg2 = ((-1.0) ** (l + idx))[:, None]
        assert np.abs(Rm[l] - sg2 * D[:, ::-1]).max() < 1e-16                 # d_mn(pi-b) = (-1)^{l+m} d_{m,-n}(b)


def test_E_R_T_agree(orc):
    L = 16
    for beta in (LD(0.02), LD(1.0), LD(2.5), LD(3.1)):
        R = orc.d_risbo(L, beta)
        for m in range(-(L - 1), L):
            for n in range(-(L - 1), L, 3):
                T = orc.d_lrec(L, m, n, beta=beta)
                for l in range(max(abs(m), abs(n)), L):
                    assert abs(T[l] - R[l][m + l, n + l]) < 2e-17
                    if l <= 10:      # the explicit alternating sum cancels digits as l grows; keep it where it is sharp
                        e = orc.d_explicit(l, m, n, beta)
                        assert abs(T[l] - e) < 1e-17 and abs(R[l][m + l, n + l] - e) < 1e-17


def test_T_vs_R_L256(orc):
    L = 256
    for beta in (np.arccos(LD(-1)) / 511, LD(0.9), LD(2.2)):
        R = orc.d_risbo(L, beta)
        worst = 0
        for (m, n) in [(0, 0), (1, 0), (17, 0), (200, 0), (255, 0), (-33, 2), (2, 2), (90, -2), (7, 7), (-7, 7), (120, -7), (3, 1)]:
            T = orc.d_lrec(L, m, n, beta=beta)
            for l in range(max(abs(m), abs(n)), L):
                worst = max(worst, abs(T[l] - R[l][m + l, n + l]))
        assert worst < 2e-16, worst


@pytest.mark.parametrize("n", [0, 2, -3])
def test_T_vs_scipy_jacobi(orc, n):
    L = 40
    for beta in (0.4, 1.7, 2.8):
        for m in range(-(L - 1), L, 5):
            T = orc.d_lrec(L, m, n, beta=LD(beta))
            for l in range(max(abs(m), abs(n)), L):
                want = jacobi_d(l, m, n, beta)
                assert abs(float(T[l]) - want) < 2e-12 * max(1.0, abs(want)), (l, m, n, beta)


def test_T_extreme_range_vs_mpmath(orc):
    """Exponent tracking: start values ~ 1e-3000 must grow back to the right O(1) values (Eq. 22 via mpmath)."""
    mp.mp.dps = 60
    L = 1200
    for (m, n, beta) in [(1100, 0, 0.05), (900, 2, 0.3), (-1000, -2, 3.0), (600, 7, 0.5)]:
        T = orc.d_lrec(L, m, n, beta=LD(beta))
        # beta as the long double actually used
        b = mp.mpf(float(LD(beta))) + mp.mpf(float(LD(beta) - LD(float(LD(beta)))))
        for l in (max(abs(m), abs(n)), max(abs(m), abs(n)) + 1, 1150, 1199):
            want = jacobi_d_mp(l, m, n, b)
            got = mp.mpf(float(T[l]))
            if abs(want) > mp.mpf(10) ** -280:
                assert abs(got - want) <= abs(want) * mp.mpf(10) ** -13, (l, m, n, beta, got, want)
            else:
                assert abs(got) < 1e-270


def test_start_value_eq27(orc):
    """Eq. 27 as mantissa*2^e against 60-digit mpmath, including |d| ~ 1e-35000."""
    mp.mp.dps = 60
    for (l, k, beta) in [(5, 2, 0.9), (1023, 0, 0.01), (1023, -2, 3.1), (8191, 0, math.pi / 16383), (8191, 7, 2.0), (300, -7, 1.0)]:
        mant, e2 = orc.d_top(l, k, LD(beta))
        b = mp.mpf(beta)
        want = mp.sqrt(mp.factorial(2 * l) / (mp.factorial(l + k) * mp.factorial(l - k))) * (-mp.sin(b / 2)) ** (l - k) * mp.cos(b / 2) ** (l + k)
        got = mp.mpf(float(mant)) * mp.mpf(2) ** e2
        assert abs(got - want) <= abs(want) * mp.mpf(10) ** -13, (l, k, beta)


@pytest.mark.parametrize("n", [0, 2, -5])
def test_eq24_three_term_relation_in_m(orc, n):
    """The oracle never recurses in m; its output must nevertheless satisfy the paper's Eq. 24."""
    L, l = 61, 60
    for beta in (LD(0.35), LD(1.4), LD(2.9)):
        d = {m: orc.d_lrec(L, m, n, beta=beta)[l] for m in range(-l, l + 1)}
        d[l + 1] = LD(0)
        d[-l - 1] = LD(0)
        for m in range(-l, l + 1):
            lhs = (n - m * np.cos(beta)) / np.sin(beta) * d[m]
            rhs = 0.5 * np.sqrt(LD((l + m) * (l - m + 1))) * d[m - 1] + 0.5 * np.sqrt(LD((l - m) * (l + m + 1))) * d[m + 1]
            assert abs(lhs - rhs) < 1e-15, (m, n, float(beta))

"""Pins for the oracle's DH, MWSS and Gauss-Legendre samplings (SURVEY 8(f) N2; PAPER.md:314-331 Eq. 34-36, :349-381 Eq. 39-44,
:383-397 Eq. 45-46): ring positions, weights against independent closed forms / numpy's Gauss-Legendre rule, exactness of the
quadratures on the band-limit they are built for (and failure beyond), closed-form harmonics on the new grids, discrete
orthonormality, and the exact inverse -> forward round trip every sampling theorem must give."""
import numpy as np
import pytest

from paper_2311_14670_b200 import synth
from test_oracle_s2 import CLOSED, closed_form_sYlm, grid

LD = np.longdouble
PI = np.arccos(LD(-1))
MW, HEALPIX, MW_QUAD, MWSS, DH, GL, MWSS_QUAD = 0, 1, 2, 3, 4, 5, 6


def test_dh_positions_and_weights_eq34_36(orc):
    for L in (1, 2, 5, 16, 33):
        tab = orc.ring_table(DH, L)
        t = np.arange(2 * L, dtype=LD)
        theta = (2 * t + 1) * PI / (4 * L)                                     # Eq. 34
        assert len(tab["nphi"]) == 2 * L and np.all(tab["nphi"] == 2 * L - 1)    # Eq. 35
        assert np.abs(np.cos(theta) - tab["cos_theta"]).max() < 1e-18
        q = tab["weight"]
        assert abs((q * tab["nphi"]).sum() - 4 * PI) < 1e-16                    # the weights integrate 1 over the sphere
        # Eq. 36 equals Fejer's first rule on these nodes (closed form, written independently of the oracle's sine sum):
        # a_t = (1/L) (1 + 2 sum_{j=1}^{L} cos(2 j theta_t)/(1-4j^2))
        a = np.array([(1 + 2 * sum(np.cos(2 * j * th) / (1 - 4 * LD(j) * j) for j in range(1, L + 1))) / L for th in theta])
        assert np.abs(q * (2 * L - 1) / (2 * PI) - a).max() < 1e-17
        # exact for cos(k theta) sin(theta), k <= 2L-1 (a polynomial of degree < 2L in cos theta) ...
        v = q * (2 * L - 1) / (2 * PI)
        for k in range(0, 2 * L):
            want = 2 / LD(1 - k * k) if k % 2 == 0 else LD(0)
            assert abs((v * np.cos(k * theta)).sum() - want) < 1e-16, (L, k)
        # ... and not beyond
        assert abs((v * np.cos(4 * L * theta)).sum() - 2 / LD(1 - 16 * L * L)) > 1e-6


def test_gl_nodes_and_weights_vs_numpy_leggauss(orc):
    """Reading R22: Eq. 46 as printed is not the Gauss-Legendre weight; the oracle uses 2/((1-x^2) P_L'(x)^2) q_Phi."""
    for L in (1, 2, 3, 8, 33, 128):
        tab = orc.ring_table(GL, L)
        x, w = np.polynomial.legendre.leggauss(L)
        assert np.all(tab["nphi"] == 2 * L - 1)                                   # Eq. 45
        assert np.abs(np.asarray(tab["cos_theta"], float) - x[::-1]).max() < 5e-15          # north to south
        v = tab["weight"] * (2 * L - 1) / (2 * PI)
        assert np.abs(np.asarray(v, float) - w[::-1]).max() < 3e-14      # numpy's own double-precision accuracy
        assert abs(v.sum() - 2) < 1e-17
        # Gauss rule: exact for polynomials of degree <= 2L-1 in x
        xs = tab["cos_theta"]
        for d in range(0, 2 * L):
            want = LD(2) / (d + 1) if d % 2 == 0 else LD(0)
            assert abs((v * xs ** d).sum() - want) < 1e-16, (L, d)
        assert abs((v * xs ** (2 * L)).sum() - LD(2) / (2 * L + 1)) > 1e-12 or L > 20
        z = tab["cos_theta"]
        assert np.abs(z + z[::-1]).max() < 1e-18                                  # symmetric about the equator


def test_mwss_positions_and_weights_eq39_44(orc):
    for L in (2, 5, 16):
        tab = orc.ring_table(MWSS, L)
        assert len(tab["nphi"]) == L + 1 and np.all(tab["nphi"] == 2 * L)         # Eq. 39-40
        t = np.arange(L + 1, dtype=LD)
        assert np.abs(np.cos(2 * PI * t / (2 * L)) - tab["cos_theta"]).max() < 1e-18
        assert tab["sin_theta"][0] == 0 and tab["sin_theta"][-1] == 0             # both poles are rings
        # quadrature grid of band-limit 2L: 2L+1 rings theta'_u = 2 pi u/(4L), weights Eq. 43-44 at T = 4L
        q = orc.ring_table(MWSS_QUAD, L)
        v = q["weight"] * (2 * L) / (2 * PI)
        u = np.arange(2 * L + 1, dtype=LD)
        theta = 2 * PI * u / (4 * L)
        assert np.abs(np.cos(theta) - q["cos_theta"]).max() < 1e-18
        assert abs(v.sum() - 2) < 1e-17
        for k in range(0, 2 * L):      # exact for even integrands of degree <= 2L-1 on the theta circle
            want = 2 / LD(1 - k * k) if k % 2 == 0 else LD(0)
            assert abs((v * np.cos(k * theta)).sum() - want) < 1e-17, (L, k)
        assert abs((v * np.cos(4 * L * theta)).sum() - 2 / LD(1 - 16 * L * L)) > 1e-6


@pytest.mark.parametrize("sampling,L", [(MWSS, 6), (DH, 6), (GL, 6)])
def test_inverse_of_unit_coefficient_is_closed_form_sYlm(orc, sampling, L):
    t, p = grid(orc, sampling, L)
    for (s, l, m) in CLOSED:
        flm = np.zeros((L, 2 * L - 1), complex)
        flm[l, m + L - 1] = 1.0
        f = orc.s2_inverse(L, s, sampling, flm).ravel()
        assert np.abs(f - closed_form_sYlm(s, l, m, t, p)).max() < 2e-15, (sampling, s, l, m)


@pytest.mark.parametrize("sampling,L", [(MWSS, 6), (DH, 6), (GL, 6)])
def test_forward_of_closed_form_sYlm_is_delta(orc, sampling, L):
    """Discrete orthonormality on each sampling theorem's grid: forward(samples of sY_l'm') = delta."""
    t, p = grid(orc, sampling, L)
    for (s, l, m) in CLOSED:
        f = closed_form_sYlm(s, l, m, t, p).reshape(orc.map_shape(sampling, L))
        flm = orc.s2_forward(L, s, sampling, f)
        want = np.zeros_like(flm)
        want[l, m + L - 1] = 1
        assert np.abs(flm - want).max() < 2e-14, (sampling, s, l, m)


@pytest.mark.parametrize("sampling", [MWSS, DH, GL])
@pytest.mark.parametrize("L,spin", [(1, 0), (2, 0), (5, 0), (12, 0), (12, 1), (12, 2), (12, -3), (33, 2), (32, -1)])
def test_round_trip_is_exact(orc, sampling, L, spin):
    """Sampling theorems: forward(inverse(flm)) = flm to rounding."""
    flm = synth.random_flm(L, spin, seed=L + spin)
    f = orc.s2_inverse(L, spin, sampling, flm)
    assert f.shape == orc.map_shape(sampling, L)
    back = orc.s2_forward(L, spin, sampling, f)
    assert np.abs(back - flm).max() < 3e-15 * L


@pytest.mark.parametrize("spin", [0, 1, -2])
def test_separable_equals_unseparated_definition(orc, spin):
    L = 7
    flm = synth.random_flm(L, spin, seed=3)
    for sampling in (MWSS, DH, GL):
        a = orc.s2_inverse(L, spin, sampling, flm)
        b = orc.s2_inverse(L, spin, sampling, flm, direct=True)
        assert np.abs(a - b).max() < 5e-15


def test_all_samplings_agree_on_the_same_function(orc):
    """One band-limited function sampled on five grids: every sampling theorem's forward transform recovers the same coefficients,
    and the maps agree where the grids share a point (MWSS ring t and DH: none; MW ring t vs MWSS: none in general -- so compare
    through the coefficients only) and at the poles of MWSS: f(0, phi) = c e^{-i s phi}, f(pi, phi) = c' e^{+i s phi} (Eq. 28-29)."""
    L, spin = 9, 2
    flm = synth.random_flm(L, spin, seed=21)
    for sampling in (MW, MWSS, DH, GL):
        back = orc.s2_forward(L, spin, sampling, orc.s2_inverse(L, spin, sampling, flm))
        assert np.abs(back - flm).max() < 1e-13
    f = orc.s2_inverse(L, spin, MWSS, flm)
    n = 2 * L
    ph = 2 * np.pi * np.arange(n) / n
    north, south = np.fft.fft(f[0]) / n, np.fft.fft(f[-1]) / n
    keepn, keeps = (-spin) % n, spin % n                      # only m = -s survives at theta = 0, only m = +s at theta = pi
    assert np.abs(np.delete(north, keepn)).max() < 1e-15 and np.abs(np.delete(south, keeps)).max() < 1e-15
    assert abs(north[keepn]) > 1e-3 and abs(south[keeps]) > 1e-3
    del ph


def test_theta_forward_columns_matches_full_forward(orc):
    """orc_s2_theta_forward_columns (Eq. 30 alone) on the weighted ring DFT of a DH map = the pinned forward transform."""
    L, spin = 10, 1
    f = synth.random_map(orc.map_shape(DH, L), seed=2)
    tab = orc.ring_table(DH, L)
    ms = np.arange(-(L - 1), L)
    Fm = np.fft.fft(f, axis=1)                                       # sum_p f e^{-i m phi_p}, bins m mod (2L-1)
    W = np.stack([Fm[:, m % (2 * L - 1)] * np.asarray(tab["weight"], float) for m in ms])
    cols = orc.s2_theta_forward_columns(L, spin, DH, W, ms)
    full = orc.s2_forward(L, spin, DH, f)
    assert np.abs(cols.T - full).max() < 1e-14

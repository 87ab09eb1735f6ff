"""Pins for the oracle's S^2 transforms: closed-form harmonics, scipy, un-separated sums, quadrature exactness,
exact MW round trip (sampling theorem), HEALPix geometry/normalisation.  SURVEY.md 8(c) pins 1, 6-9."""
import os

import numpy as np
import pytest
from scipy.special import sph_harm_y

from paper_2311_14670_b200 import synth

LD = np.longdouble
HERE = os.path.dirname(os.path.abspath(__file__))


def grid(orc, sampling, L, nside=0):
    """(theta, phi) of every sample in map order, in double."""
    tab = orc.ring_table(sampling, L, nside)
    th, ph = [], []
    for ct, st, n, p0 in zip(tab["cos_theta"], tab["sin_theta"], tab["nphi"], tab["phi0"]):
        t = float(np.arctan2(st, ct))
        th.append(np.full(n, t))
        ph.append(float(p0) + 2 * np.pi * np.arange(n) / n)
    return np.concatenate(th), np.concatenate(ph)


def closed_form_sYlm(s, l, m, t, p):
    """Closed forms, spin 0 l<=3 and spin 1/2 lowest l (standard tables; SURVEY.md 8(c) pin 1)."""
    c, sn, e = np.cos(t), np.sin(t), np.exp(1j * m * p)
    pi = np.pi
    if s == 0:
        tbl = {
            (0, 0): 1 / np.sqrt(4 * pi) + 0 * t, (1, 0): np.sqrt(3 / (4 * pi)) * c,
            (1, 1): -np.sqrt(3 / (8 * pi)) * sn, (1, -1): np.sqrt(3 / (8 * pi)) * sn,
            (2, 0): np.sqrt(5 / (16 * pi)) * (3 * c * c - 1),
            (2, 1): -np.sqrt(15 / (8 * pi)) * sn * c, (2, -1): np.sqrt(15 / (8 * pi)) * sn * c,
            (2, 2): np.sqrt(15 / (32 * pi)) * sn * sn, (2, -2): np.sqrt(15 / (32 * pi)) * sn * sn,
            (3, 0): np.sqrt(7 / (16 * pi)) * (5 * c ** 3 - 3 * c),
            (3, 1): -np.sqrt(21 / (64 * pi)) * sn * (5 * c * c - 1), (3, -1): np.sqrt(21 / (64 * pi)) * sn * (5 * c * c - 1),
            (3, 2): np.sqrt(105 / (32 * pi)) * sn * sn * c, (3, -2): np.sqrt(105 / (32 * pi)) * sn * sn * c,
            (3, 3): -np.sqrt(35 / (64 * pi)) * sn ** 3, (3, -3): np.sqrt(35 / (64 * pi)) * sn ** 3,
        }
        return tbl[(l, m)] * e
    if s == 1:
        tbl = {(1, 0): np.sqrt(3 / (8 * pi)) * sn, (1, 1): -np.sqrt(3 / (16 * pi)) * (1 - c), (1, -1): -np.sqrt(3 / (16 * pi)) * (1 + c)}
        return tbl[(l, m)] * e
    if s == 2:
        tbl = {(2, 0): np.sqrt(15 / (32 * pi)) * sn * sn, (2, 1): -np.sqrt(5 / (16 * pi)) * sn * (1 - c),
               (2, -1): -np.sqrt(5 / (16 * pi)) * sn * (1 + c), (2, 2): np.sqrt(5 / (64 * pi)) * (1 - c) ** 2,
               (2, -2): np.sqrt(5 / (64 * pi)) * (1 + c) ** 2}
        return tbl[(l, m)] * e
    raise KeyError


CLOSED = [(0, l, m) for l in range(4) for m in range(-l, l + 1)] + [(1, 1, m) for m in (-1, 0, 1)] + [(2, 2, m) for m in range(-2, 3)]


@pytest.mark.parametrize("sampling,L,nside", [(0, 6, 0), (1, 5, 2)])
def test_inverse_of_unit_coefficient_is_closed_form_sYlm(orc, sampling, L, nside):
    t, p = grid(orc, sampling, L, nside)
    for (s, l, m) in CLOSED:
        flm = np.zeros((L, 2 * L - 1), complex)
        flm[l, m + L - 1] = 1.0
        f = orc.s2_inverse(L, s, sampling, flm, nside=nside).ravel()
        want = closed_form_sYlm(s, l, m, t, p)
        assert np.abs(f - want).max() < 2e-15, (s, l, m)
        if s != 0:  # negative spin through  conj(sY_lm) = (-1)^{s+m} (-s)Y_{l,-m}
            flm2 = np.zeros_like(flm)
            flm2[l, -m + L - 1] = 1.0
            f2 = orc.s2_inverse(L, -s, sampling, flm2, nside=nside).ravel()
            assert np.abs(f2 - (-1.0) ** (s + m) * np.conj(want)).max() < 2e-15, (-s, l, -m)


def test_inverse_vs_scipy_spin0(orc):
    L = 40
    flm = synth.random_flm(L, 0, seed=11)
    t, p = grid(orc, 0, L)
    want = np.zeros(t.shape, complex)
    for l in range(L):
        for m in range(-l, l + 1):
            want += flm[l, m + L - 1] * sph_harm_y(l, m, t, p)
    f = orc.s2_inverse(L, 0, 0, flm).ravel()
    assert np.abs(f - want).max() < 5e-13 * np.abs(want).max()


@pytest.mark.parametrize("spin", [0, 1, -2])
def test_separable_equals_unseparated_definition(orc, spin):
    L = 7
    flm = synth.random_flm(L, spin, seed=3)
    for sampling, nside in ((0, 0), (1, 2)):
        a = orc.s2_inverse(L, spin, sampling, flm, nside=nside)
        b = orc.s2_inverse(L, spin, sampling, flm, nside=nside, direct=True)
        assert np.abs(a - b).max() < 5e-15
    f = synth.random_map((12 * 4,), seed=5)
    a = orc.s2_forward(L, spin, 1, f, nside=2)
    b = orc.s2_forward(L, spin, 1, f, nside=2, direct=True)
    assert np.abs(a - b).max() < 5e-15


def test_mw_quadrature_weights_exact(orc):
    """sum_u v_u cos(k theta'_u) = int_0^pi cos(k t) sin t dt = 2/(1-k^2) (k even), 0 (k odd), for |k| <= 2L-1."""
    for L in (4, 9, 32):
        tab = orc.ring_table(2, L)
        v = tab["weight"] * (2 * L - 1) / (2 * np.arccos(LD(-1)))     # strip q_phi = 2pi/(2L-1)
        assert len(v) == 2 * L and abs(v.sum() - 2) < 1e-17
        u = np.arange(2 * L, dtype=LD)
        theta = np.arccos(LD(-1)) * (2 * u + 1) / (4 * L - 1)
        assert np.abs(np.cos(theta) - tab["cos_theta"]).max() < 1e-18
        for k in range(0, 2 * L):
            want = 2 / LD(1 - k * k) if k % 2 == 0 else LD(0)
            assert abs((v * np.cos(k * theta)).sum() - want) < 1e-17, (L, k)
        # ... and it is NOT exact beyond the band-limit it was built for
        assert abs((v * np.cos(4 * L * theta)).sum() - 2 / LD(1 - 16 * L * L)) > 1e-6


@pytest.mark.parametrize("L,spin", [(5, 0), (12, 0), (12, 1), (12, 2), (12, -3), (33, 2), (32, -1)])
def test_mw_round_trip_is_exact(orc, L, spin):
    """Sampling theorem: forward(inverse(flm)) = flm to rounding."""
    flm = synth.random_flm(L, spin, seed=L + spin)
    f = orc.s2_inverse(L, spin, 0, flm)
    back = orc.s2_forward(L, spin, 0, f)
    assert np.abs(back - flm).max() < 3e-15 * L


def test_forward_of_closed_form_sYlm_is_delta(orc):
    """Discrete orthonormality on the MW grid (Eq. 2 + sampling theorem): forward(samples of sY_l'm') = delta."""
    L = 6
    t, p = grid(orc, 0, L)
    for (s, l, m) in CLOSED:
        f = closed_form_sYlm(s, l, m, t, p).reshape(L, 2 * L - 1)
        flm = orc.s2_forward(L, s, 0, f)
        want = np.zeros_like(flm)
        want[l, m + L - 1] = 1
        assert np.abs(flm - want).max() < 1e-14, (s, l, m)


def test_columns_and_rings_subsets_match_full(orc):
    L, spin = 10, 2
    flm = synth.random_flm(L, spin, seed=2)
    f = orc.s2_inverse(L, spin, 0, flm)
    rows = orc.s2_inverse_rings(L, spin, 0, flm, [0, 4, 9])
    for r, row in zip([0, 4, 9], rows):
        assert np.array_equal(row, f[r])
    ms = [-9, -2, 0, 3]
    cols = orc.s2_forward_columns(L, spin, 0, f, ms)
    full = orc.s2_forward(L, spin, 0, f)
    for i, m in enumerate(ms):
        assert np.array_equal(cols[i], full[:, m + L - 1])


def test_theta_step_columns_is_ring_dft_of_map(orc):
    """Eq. 32: the map's ring DFT equals F_m(theta) of Eq. 33 (ties theta_inverse_columns to the pinned inverse)."""
    L, spin = 9, 1
    flm = synth.random_flm(L, spin, seed=8)
    f = orc.s2_inverse(L, spin, 0, flm)
    ms = np.arange(-(L - 1), L)
    F = orc.s2_theta_inverse_columns(L, spin, 0, flm, ms)          # [m, ring]
    Fd = np.fft.fft(f, axis=1) / (2 * L - 1)                         # phi_p = 2 pi p/(2L-1)
    for i, m in enumerate(ms):
        assert np.abs(F[i] - Fd[:, m % (2 * L - 1)]).max() < 1e-14


def test_healpix_geometry(orc):
    tab = orc.ring_table(1, 0, 1)
    # nside = 1: 12 pixels on rings z = 2/3, 0, -2/3; four per ring; phi = pi/4 + k pi/2, k pi/2, pi/4 + k pi/2.
    assert list(tab["nphi"]) == [4, 4, 4]
    assert np.allclose(np.asarray(tab["cos_theta"], float), [2 / 3, 0, -2 / 3], atol=1e-18)
    assert np.allclose(np.asarray(tab["phi0"], float), [np.pi / 4, 0, np.pi / 4])
    for nside in (2, 4, 16, 64):
        tab = orc.ring_table(1, 0, nside)
        assert len(tab["nphi"]) == 4 * nside - 1
        assert tab["nphi"].sum() == 12 * nside * nside == orc.num_pixels(1, 0, nside)
        z = tab["cos_theta"]
        assert np.abs(z + z[::-1]).max() == 0 and z[2 * nside - 1] == 0
        assert np.all(np.diff(z) < 0)
        assert abs((tab["weight"] * tab["nphi"]).sum() - 4 * np.arccos(LD(-1))) < 1e-17
        assert np.all(tab["nphi"][:nside - 1] == 4 * np.arange(1, nside)) and np.all(tab["nphi"][nside - 1:3 * nside] == 4 * nside)
        # ring pixel-centre heights follow equal-area rows: consecutive belt rings are 2/(3 nside) apart in z
        assert np.allclose(np.asarray(np.diff(z[nside - 1:3 * nside]), float), -2 / (3 * nside), atol=1e-17)


def test_healpix_forward_normalisation_and_real_maps(orc):
    nside, L = 4, 8
    c = 1.7
    flm = orc.s2_forward(L, 0, 1, np.full(12 * nside * nside, c, complex), nside=nside)
    assert abs(flm[0, L - 1] - c * np.sqrt(4 * np.pi)) < 1e-14          # sum_pix (4pi/Npix) c Y_00
    flm_r = synth.random_flm(L, 0, seed=4, real=True)
    f = orc.s2_inverse(L, 0, 1, flm_r, nside=nside)
    assert np.abs(f.imag).max() < 1e-15
    back = orc.s2_forward(L, 0, 1, f, nside=nside)
    # no sampling theorem: the single-pass round trip is only approximate
    rel = np.abs(back - flm_r).max() / np.abs(flm_r).max()
    assert 1e-4 < rel < 0.3


def _paper_table(name):
    out = {}
    for line in open(os.path.join(HERE, "golden", "paper_tables_roundtrip.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t, L, e = line.split()
        if t == name:
            out[int(L)] = float(e)
    return out


def test_round_trip_error_is_below_paper_table1(orc):
    """Table 1: the paper's fp64 MW round-trip errors are 3.6e-16 (L=8) ... 1.2e-15 (L=64).
    The oracle works in long double, so its own round trip must sit below those figures (it is the reference the
    fp64 GPU path is judged against; the GPU test compares its error with the same table)."""
    tab = _paper_table("sht")
    for L in (8, 16, 32, 64):
        errs = []
        for seed in range(3):
            flm = synth.random_flm(L, 0, seed=100 + seed)
            back = orc.s2_forward(L, 0, 0, orc.s2_inverse(L, 0, 0, flm))
            sup = flm != 0
            errs.append(np.abs(back - flm)[sup].mean())
        e = float(np.mean(errs))
        assert e < tab[L] / 3, (L, e, tab[L])


def test_healpix_iterative_refinement(orc):
    """HEALPix transforms are approximate and "iterations are usually performed".  The iteration
    flm <- flm + F (f - F^-1 flm) (reading R24) must (a) reduce to the plain forward at niter = 0, (b) shrink the map residual
    |f - F^-1 flm| at every step, and (c) move the coefficients of a band-limited map toward the generating ones."""
    nside, L = 8, 16
    flm = synth.random_flm(L, 0, seed=6, sigma=synth.SIGMA_RED, real=True)
    f = orc.s2_inverse(L, 0, 1, flm, nside=nside)
    assert np.array_equal(orc.s2_forward_iter(L, 0, 1, f, 0, nside=nside), orc.s2_forward(L, 0, 1, f, nside=nside))
    errs, res = [], []
    for it in range(4):
        c = orc.s2_forward_iter(L, 0, 1, f, it, nside=nside)
        errs.append(np.abs(c - flm).max() / np.abs(flm).max())
        res.append(np.abs(f - orc.s2_inverse(L, 0, 1, c, nside=nside)).max())
    assert all(b < a for a, b in zip(res, res[1:])) and all(b < a for a, b in zip(errs, errs[1:]))
    assert errs[3] < errs[0] / 20
    # one step written out by hand from the pinned F and F^-1
    c0 = orc.s2_forward(L, 0, 1, f, nside=nside)
    c1 = c0 + orc.s2_forward(L, 0, 1, f - orc.s2_inverse(L, 0, 1, c0, nside=nside), nside=nside)
    assert np.abs(orc.s2_forward_iter(L, 0, 1, f, 1, nside=nside) - c1).max() < 1e-16


@pytest.mark.parametrize("spin", [0, 2, -1])
def test_healpix_forward_converges_to_the_generating_coefficients(orc, spin):
    """HEALPix has no sampling theorem, so nothing fixes the forward transform's values exactly -- but its quadrature
    (equal-area pixels, weight 4 pi / Npix) is a consistent rule: for a fixed band-limited field the forward of
    the synthesised map must converge to the GENERATING coefficients, every (l, m) and every spin, at the second order of the
    pixel size, i.e. the error falls 4x per doubling of nside.  A wrong phase convention, ring offset, weight or m-folding in the
    forward path does not converge (or converges to something else); this pins its absolute values to a truth outside the oracle."""
    L = 8
    flm = synth.random_flm(L, spin, seed=21 + spin)
    errs = []
    for nside in (4, 8, 16, 32):
        f = orc.s2_inverse(L, spin, 1, flm, nside=nside)
        back = orc.s2_forward(L, spin, 1, f, nside=nside)
        errs.append(np.abs(back - flm).max() / np.abs(flm).max())
    ratios = [a / b for a, b in zip(errs, errs[1:])]
    assert errs[0] < 0.1 and errs[-1] < 1e-3, errs
    assert all(3.5 < r < 6.0 for r in ratios) and abs(ratios[-1] - 4.0) < 0.1, ratios

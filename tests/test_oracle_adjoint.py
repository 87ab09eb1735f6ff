"""Pins for the oracle's adjoint transforms (Sec. 5.3).  The adjoints are written as plain
conjugate-transposed sums; what pins them from outside: the dot-product identity against the (separately pinned) forward and
inverse transforms on random vectors, Eq. 52 F^H = Q F^-1 and Eq. 58 F^-H = F Q^-1 on the direct-quadrature samplings, and an
explicit matrix transpose at tiny L."""
import numpy as np
import pytest

from paper_2311_14670_b200 import synth

MW, HEALPIX, MWSS, DH, GL = 0, 1, 3, 4, 5
CASES = [(MW, 0), (MWSS, 0), (DH, 0), (GL, 0), (HEALPIX, 4)]


def rand_coef(L, spin, seed):
    return synth.random_flm(L, spin, seed=seed)


def rand_map(orc, sampling, L, nside, seed):
    return synth.random_map(orc.map_shape(sampling, L, nside), seed=seed)


def ring_weights(orc, sampling, L, nside):
    """q(theta, phi) per sample in map order (direct-quadrature samplings)."""
    tab = orc.ring_table(sampling, L, nside)
    return np.concatenate([np.full(n, float(w)) for n, w in zip(tab["nphi"], tab["weight"])])


@pytest.mark.parametrize("sampling,nside", CASES)
@pytest.mark.parametrize("L,spin", [(7, 0), (12, 2), (12, -1), (20, 0)])
def test_dot_product_identities(orc, sampling, nside, L, spin):
    """<F x, y> = <x, F^H y> and <F^-1 c, g> = <c, F^-H g> for random x, y (not band-limited: the identity is about matrices)."""
    x = rand_map(orc, sampling, L, nside, 1)
    y = rand_coef(L, spin, 2)
    a = np.vdot(y, orc.s2_forward(L, spin, sampling, x, nside=nside))
    b = np.vdot(orc.s2_forward_adjoint(L, spin, sampling, y, nside=nside), x)
    assert abs(a - b) < 1e-13 * abs(a)
    c = rand_coef(L, spin, 3)
    g = rand_map(orc, sampling, L, nside, 4)
    a = np.vdot(g, orc.s2_inverse(L, spin, sampling, c, nside=nside))
    b = np.vdot(orc.s2_inverse_adjoint(L, spin, sampling, g, nside=nside), c)
    assert abs(a - b) < 1e-13 * abs(a)


@pytest.mark.parametrize("sampling,nside", [(DH, 0), (GL, 0), (HEALPIX, 2), (HEALPIX, 4)])
@pytest.mark.parametrize("spin", [0, 2])
def test_eq52_and_eq58_on_direct_quadrature_samplings(orc, sampling, nside, spin):
    """Eq. 52: F^H = Q F^-1;  Eq. 58: F^-H = F Q^-1 -- against the pinned forward / inverse transforms."""
    L = 10
    q = ring_weights(orc, sampling, L, nside)
    shape = orc.map_shape(sampling, L, nside)
    y = rand_coef(L, spin, 5)
    lhs = orc.s2_forward_adjoint(L, spin, sampling, y, nside=nside)
    rhs = q.reshape(shape) * orc.s2_inverse(L, spin, sampling, y, nside=nside)
    assert np.abs(lhs - rhs).max() < 1e-15 * np.abs(rhs).max()
    g = rand_map(orc, sampling, L, nside, 6)
    lhs = orc.s2_inverse_adjoint(L, spin, sampling, g, nside=nside)
    rhs = orc.s2_forward(L, spin, sampling, g / q.reshape(shape), nside=nside)
    assert np.abs(lhs - rhs).max() < 1e-13 * np.abs(rhs).max()


@pytest.mark.parametrize("sampling", [MW, MWSS])
def test_adjoint_is_the_conjugate_transpose_of_the_explicit_matrix(orc, sampling):
    """Tiny L: build the matrix of the forward transform column by column from unit maps and compare F^H with its transpose."""
    L, spin = 4, 1
    shape = orc.map_shape(sampling, L)
    npix = int(np.prod(shape))
    A = np.zeros((L * (2 * L - 1), npix), complex)
    for j in range(npix):
        e = np.zeros(npix, complex); e[j] = 1
        A[:, j] = orc.s2_forward(L, spin, sampling, e.reshape(shape)).ravel()
    y = rand_coef(L, spin, 9)
    got = orc.s2_forward_adjoint(L, spin, sampling, y).ravel()
    assert np.abs(got - A.conj().T @ y.ravel()).max() < 1e-15
    B = np.zeros((npix, L * (2 * L - 1)), complex)
    for j in range(L * (2 * L - 1)):
        e = np.zeros(L * (2 * L - 1), complex); e[j] = 1
        B[:, j] = orc.s2_inverse(L, spin, sampling, e.reshape(L, 2 * L - 1)).ravel()
    g = synth.random_map(shape, seed=3)
    got = orc.s2_inverse_adjoint(L, spin, sampling, g).ravel()
    want = B.conj().T @ g.ravel()
    el = np.repeat(np.arange(L), 2 * L - 1); m = np.tile(np.arange(-(L - 1), L), L)
    sup = (np.abs(m) <= el) & (el >= abs(spin))
    assert np.abs(got - want)[sup].max() < 1e-14 and np.all(got[~sup] == 0)


@pytest.mark.parametrize("L,N", [(5, 1), (6, 3), (9, 4), (8, 8)])
def test_so3_dot_product_identities(orc, L, N):
    """Wigner transforms (Eq. 15-18): <W x, y> = <x, W^H y> and <W^-1 c, g> = <c, W^-H g> on random (not band-limited) arrays, against the
    separately pinned so3_forward / so3_inverse.  A wrong l-scaling, gamma sign, spin sign or slab order in the transposed chain breaks it."""
    shape = (2 * N - 1, L, 2 * L - 1)
    x = synth.random_map(shape, seed=1)
    y = synth.random_flmn(L, N, seed=2)
    a = np.vdot(y, orc.so3_forward(L, N, x))
    b = np.vdot(orc.so3_forward_adjoint(L, N, y), x)
    assert abs(a - b) < 1e-13 * abs(a)
    c = synth.random_flmn(L, N, seed=3)
    g = synth.random_map(shape, seed=4)
    a = np.vdot(g, orc.so3_inverse(L, N, c))
    b = np.vdot(orc.so3_inverse_adjoint(L, N, g), c)
    assert abs(a - b) < 1e-13 * abs(a)
    # coefficients outside the support (l < |n|, l < |m|) of the inverse's adjoint are zero
    out = orc.so3_inverse_adjoint(L, N, g)
    el = np.arange(L)[None, :, None]
    m = np.arange(-(L - 1), L)[None, None, :]
    n = (np.arange(2 * N - 1) - (N - 1))[:, None, None]
    assert np.all(out[(np.abs(m) > el) | (np.abs(n) > el)] == 0)

"""Pins for the oracle's Wigner (SO(3)) transforms: closed-form D^1, relation to spin transforms (Eq. 15-18),
exact round trip on the MW-SO3 sampling theorem.  SURVEY.md 8(c) pins 1, 6 and readings R1, R2, R19."""
import numpy as np
import pytest

from paper_2311_14670_b200 import synth


def so3_grid(L, N):
    a = 2 * np.pi * np.arange(2 * L - 1) / (2 * L - 1)
    b = np.pi * (2 * np.arange(L) + 1) / (2 * L - 1)
    g = 2 * np.pi * np.arange(2 * N - 1) / (2 * N - 1)
    return a, b, g


def d1(m, n, b):
    """Closed-form d^1_mn (Varshalovich tables)."""
    c, s = np.cos(b), np.sin(b)
    tbl = {(1, 1): (1 + c) / 2, (1, 0): -s / np.sqrt(2), (1, -1): (1 - c) / 2,
           (0, 1): s / np.sqrt(2), (0, 0): c, (0, -1): -s / np.sqrt(2),
           (-1, 1): (1 - c) / 2, (-1, 0): s / np.sqrt(2), (-1, -1): (1 + c) / 2}
    return tbl[(m, n)]


def test_inverse_of_unit_coefficient_is_conj_D(orc):
    """Eq. 13: a single f^l_mn = 1 synthesises (2l+1)/(8 pi^2) conj(D^l_mn) with D of Eq. 10."""
    L, N = 4, 2
    a, b, g = so3_grid(L, N)
    for m in (-1, 0, 1):
        for n in (-1, 0, 1):
            c = np.zeros((2 * N - 1, L, 2 * L - 1), complex)
            c[n + N - 1, 1, m + L - 1] = 1
            f = orc.so3_inverse(L, N, c)
            want = 3 / (8 * np.pi ** 2) * np.exp(1j * n * g)[:, None, None] * d1(m, n, b)[None, :, None] * np.exp(1j * m * a)[None, None, :]
            assert np.abs(f - want).max() < 1e-15, (m, n)
    c = np.zeros((2 * N - 1, L, 2 * L - 1), complex)
    c[N - 1, 0, L - 1] = 1
    assert np.abs(orc.so3_inverse(L, N, c) - 1 / (8 * np.pi ** 2)).max() < 1e-16


@pytest.mark.parametrize("L,N", [(6, 1), (8, 3), (9, 9), (16, 5)])
def test_round_trip_is_exact(orc, L, N):
    c = synth.random_flmn(L, N, seed=L * 10 + N)
    back = orc.so3_forward(L, N, orc.so3_inverse(L, N, c))
    assert np.abs(back - c).max() < 3e-15 * L


def test_wigner_inverse_is_a_sum_of_spin_transforms(orc):
    """Eq. 17-18 (reading R1): f = sum_n e^{i n gamma} f_n,
    f_n = (-1)^n sum_lm sqrt((2l+1)/(16 pi^3)) f^l_mn  (-n)Y_lm(beta, alpha)  -- ties SO(3) to the pinned S^2 inverse."""
    L, N = 10, 4
    c = synth.random_flmn(L, N, seed=5)
    f = orc.so3_inverse(L, N, c)
    _, _, g = so3_grid(L, N)
    el = np.arange(L)[:, None]
    want = np.zeros_like(f)
    for n in range(-(N - 1), N):
        flm = (-1.0) ** n * np.sqrt((2 * el + 1) / (16 * np.pi ** 3)) * c[n + N - 1]
        fn = orc.s2_inverse(L, -n, 0, flm)
        want += np.exp(1j * n * g)[:, None, None] * fn[None]
    assert np.abs(f - want).max() < 1e-14 * np.abs(want).max()


def test_forward_is_scaled_spin_transform(orc):
    """Eq. 15-16: f^l_mn = (-1)^n sqrt(4pi/(2l+1)) * [spin -n forward SHT of f_n]."""
    L, N = 9, 3
    f = orc.so3_inverse(L, N, synth.random_flmn(L, N, seed=9))
    got = orc.so3_forward(L, N, f)
    _, _, g = so3_grid(L, N)
    el = np.arange(L)[:, None]
    for n in range(-(N - 1), N):
        fn = (2 * np.pi / (2 * N - 1)) * np.tensordot(np.exp(-1j * n * g), f, axes=(0, 0))
        flm = orc.s2_forward(L, -n, 0, fn)
        want = (-1.0) ** n * np.sqrt(4 * np.pi / (2 * el + 1)) * flm
        assert np.abs(got[n + N - 1] - want).max() < 1e-14


def test_coefficients_outside_support_are_ignored_and_zeroed(orc):
    L, N = 6, 3
    c = synth.random_flmn(L, N, seed=1)
    junk = c.copy()
    junk[0, 0, :] = 5.0      # n = -2 at l = 0: outside |n| <= l
    assert np.array_equal(orc.so3_inverse(L, N, junk), orc.so3_inverse(L, N, c))
    back = orc.so3_forward(L, N, orc.so3_inverse(L, N, c))
    assert np.all(back[0, 0, :] == 0) and np.all(back[0, 1, :] == 0)

"""Seeded synthetic inputs shared by the tests, bench.py and smoke() -- data only, none of the method's arithmetic.

The paper measures on "random band-limited functions"; these generators stand in for them with
the shapes / value distributions of BASELINE.json's configs (recipe: DESIGN.md "Synthetic inputs").  Arrays are
drawn in the dense row-major order of the public layouts (flm[L][2L-1], flmn[2N-1][L][2L-1]) from
numpy.random.default_rng(seed) (PCG64), then entries outside the coefficient support are zeroed.
"""
import numpy as np

SIGMA_UNIT = "unit"            # sigma_l = 1                           (configs 1, 4)
SIGMA_CMB = "1/sqrt(l(l+1))"   # sigma_l^2 = 1/(l(l+1)), l >= 2        (config 2)
SIGMA_RED = "1/(l+1)"          # sigma_l = 1/(l+1)                     (configs 3, 5)


def _sigma(L, mode):
    el = np.arange(L, dtype=np.float64)
    if mode == SIGMA_UNIT:
        return np.ones(L)
    if mode == SIGMA_CMB:
        s = np.zeros(L)
        s[2:] = 1.0 / np.sqrt(el[2:] * (el[2:] + 1.0))
        return s
    if mode == SIGMA_RED:
        return 1.0 / (el + 1.0)
    raise ValueError(mode)


def random_flm(L, spin=0, seed=0, sigma=SIGMA_UNIT, real=False):
    """Complex coefficients flm[L][2L-1] (column m+L-1), E|flm|^2 = sigma_l^2 on the support l>=|spin|, |m|<=l.

    real=True (spin 0 only): Im f_l0 = 0 and f_{l,-m} = (-1)^m conj(f_lm), i.e. the coefficients of a real map
    (PAPER.md:76).
    """
    rng = np.random.default_rng(seed)
    g = rng.standard_normal((L, 2 * L - 1, 2))
    flm = (g[..., 0] + 1j * g[..., 1]) / np.sqrt(2.0)
    flm *= _sigma(L, sigma)[:, None]
    el = np.arange(L)[:, None]
    m = np.arange(-(L - 1), L)[None, :]
    flm[(np.abs(m) > el) | (el < abs(spin))] = 0.0
    if real:
        if spin != 0:
            raise ValueError("real signals are spin 0")
        flm[:, L - 1] = flm[:, L - 1].real
        pos = flm[:, L:]                                   # m = 1..L-1
        sign = np.where(np.arange(1, L) % 2 == 0, 1.0, -1.0)[None, :]
        flm[:, :L - 1] = (sign * np.conj(pos))[:, ::-1]    # m = -(L-1)..-1
    return np.ascontiguousarray(flm)


def random_flmn(L, N, seed=0):
    """Complex Wigner coefficients flmn[2N-1][L][2L-1] = (n+N-1, l, m+L-1), unit variance on |m|,|n| <= l < L."""
    rng = np.random.default_rng(seed)
    g = rng.standard_normal((2 * N - 1, L, 2 * L - 1, 2))
    c = (g[..., 0] + 1j * g[..., 1]) / np.sqrt(2.0)
    n = np.arange(-(N - 1), N)[:, None, None]
    el = np.arange(L)[None, :, None]
    m = np.arange(-(L - 1), L)[None, None, :]
    c[(np.abs(m) > el) | (np.abs(n) > el)] = 0.0
    return np.ascontiguousarray(c)


def random_map(shape, seed=0, real=False):
    """A plain (not band-limited) random map: iid N(0,1) samples (complex: unit total variance), for forward-transform parity on
    arbitrary arrays.  Nothing is special-cased: MW maps get white noise on the theta = pi ring too (R21)."""
    rng = np.random.default_rng(seed)
    if real:
        return rng.standard_normal(shape)
    g = rng.standard_normal(tuple(shape) + (2,))
    return np.ascontiguousarray((g[..., 0] + 1j * g[..., 1]) / np.sqrt(2.0))

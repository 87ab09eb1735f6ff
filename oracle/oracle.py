"""ctypes binding of oracle/libsht_oracle.so -- argument marshalling only, no arithmetic of the method.

Layouts follow DESIGN.md / include/b200sht.h: flm[L][2L-1] (column m+L-1), MW maps f[L][2L-1], HEALPix maps
ring-ordered f[12 nside^2], SO(3) f[2N-1][L][2L-1] = (gamma, beta, alpha), flmn[2N-1][L][2L-1] = (n+N-1, l, m+L-1).
All complex arrays are numpy complex128.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

MW, HEALPIX, MW_QUAD, MWSS, DH, GL, MWSS_QUAD = 0, 1, 2, 3, 4, 5, 6

_lib = None
_LD = C.c_longdouble
_PLD = C.POINTER(C.c_longdouble)
_PD = C.POINTER(C.c_double)
_PI = C.POINTER(C.c_int)


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.orc_d_explicit.restype = None
        L.orc_d_explicit.argtypes = [C.c_int, C.c_int, C.c_int, _PLD, _PLD]
        L.orc_d_risbo.restype = None
        L.orc_d_risbo.argtypes = [C.c_int, _PLD, _PLD]
        L.orc_d_lrec.restype = None
        L.orc_d_lrec.argtypes = [C.c_int, C.c_int, C.c_int, _PLD, _PLD]
        L.orc_d_top.restype = None
        L.orc_d_top.argtypes = [C.c_int, C.c_int, _PLD, _PLD, C.POINTER(C.c_long)]
        L.orc_num_rings.restype = C.c_int
        L.orc_num_rings.argtypes = [C.c_int] * 3
        L.orc_num_pixels.restype = C.c_long
        L.orc_num_pixels.argtypes = [C.c_int] * 3
        L.orc_ring_table.restype = None
        L.orc_ring_table.argtypes = [C.c_int] * 3 + [_PLD, _PLD, _PI, _PLD, _PLD, C.POINTER(C.c_long)]
        for name in ("orc_s2_inverse", "orc_s2_forward", "orc_s2_inverse_direct", "orc_s2_forward_direct"):
            f = getattr(L, name)
            f.restype = C.c_int
            f.argtypes = [C.c_int] * 4 + [_PD, _PD]
        L.orc_s2_forward_adjoint.restype = C.c_int
        L.orc_s2_forward_adjoint.argtypes = [C.c_int] * 4 + [_PD, _PD]
        for name in ("orc_s2_inverse_rings", "orc_s2_forward_columns", "orc_s2_theta_inverse_columns", "orc_s2_theta_forward_columns",
                     "orc_s2_inverse_adjoint_columns"):
            f = getattr(L, name)
            f.restype = C.c_int
            f.argtypes = [C.c_int] * 4 + [_PD, C.c_int, _PI, _PD]
        for name in ("orc_so3_inverse", "orc_so3_forward"):
            f = getattr(L, name)
            f.restype = C.c_int
            f.argtypes = [C.c_int, C.c_int, _PD, _PD]
        L.orc_threads.restype = C.c_int
        L.orc_set_threads.argtypes = [C.c_int]
        _lib = L
    return _lib


def _pd(a):
    return a.ctypes.data_as(_PD)


def _pld(*vals):
    """long double scalars cross the ABI by pointer (ctypes would round by-value long doubles to double)."""
    a = np.array(vals, dtype=np.longdouble)
    return a, a.ctypes.data_as(_PLD)


def _c128(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    if shape is not None and tuple(a.shape) != tuple(shape):
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


def _check(rc, what):
    if rc != 0:
        raise ValueError(f"oracle: {what} rejected its arguments (rc={rc})")


def threads():
    return int(lib().orc_threads())


def set_threads(n):
    lib().orc_set_threads(int(n))


# ---- Wigner d providers -----------------------------------------------------------------------------------
def d_explicit(l, m, n, beta):
    """Provider E (Wigner's explicit sum), long double."""
    b, pb = _pld(beta)
    o, po = _pld(0)
    lib().orc_d_explicit(int(l), int(m), int(n), pb, po)
    return o[0]


def d_risbo(L, beta):
    """Provider R.  Returns list over l of (2l+1)x(2l+1) longdouble arrays indexed [m+l, n+l]."""
    tot = sum((2 * l + 1) ** 2 for l in range(L))
    buf = np.zeros(tot, dtype=np.longdouble)
    b, pb = _pld(beta)
    lib().orc_d_risbo(int(L), pb, buf.ctypes.data_as(_PLD))
    out, off = [], 0
    for l in range(L):
        k = 2 * l + 1
        out.append(buf[off:off + k * k].reshape(k, k))
        off += k * k
    return out


def d_lrec(L, m, n, beta=None, cos_half=None, sin_half=None):
    """Provider T: d^l_mn for l<L at one angle.  Give beta, or the half-angle cos/sin directly."""
    if beta is not None:
        b = np.longdouble(beta)
        cos_half, sin_half = np.cos(b / 2), np.sin(b / 2)
    out = np.zeros(L, dtype=np.longdouble)
    h, ph = _pld(cos_half, sin_half)
    lib().orc_d_lrec(int(L), int(m), int(n), ph, out.ctypes.data_as(_PLD))
    return out


def d_top(l, k, beta):
    """Eq. 27 start value d^l_{l,k}(beta) as (mantissa, exponent2)."""
    b = np.longdouble(beta)
    h, ph = _pld(np.cos(b / 2), np.sin(b / 2))
    mant, pm = _pld(0)
    e2 = C.c_long(0)
    lib().orc_d_top(int(l), int(k), ph, pm, C.byref(e2))
    return mant[0], int(e2.value)


# ---- sampling ----------------------------------------------------------------------------------------------
def num_rings(sampling, L, nside=0):
    return int(lib().orc_num_rings(sampling, L, nside))


def num_pixels(sampling, L, nside=0):
    return int(lib().orc_num_pixels(sampling, L, nside))


def ring_table(sampling, L, nside=0):
    """dict(cos_theta, sin_theta, nphi, phi0, weight, offset) for any sampling code (MW_QUAD / MWSS_QUAD: the upsampled
    quadrature grids of the MW / MWSS forward transforms)."""
    nr = num_rings(sampling, L, nside)
    ct = np.zeros(nr, np.longdouble); st = np.zeros(nr, np.longdouble)
    ph = np.zeros(nr, np.longdouble); w = np.zeros(nr, np.longdouble)
    nphi = np.zeros(nr, np.int32); off = np.zeros(nr, np.int64)
    lib().orc_ring_table(sampling, L, nside, ct.ctypes.data_as(_PLD), st.ctypes.data_as(_PLD),
                         nphi.ctypes.data_as(_PI), ph.ctypes.data_as(_PLD), w.ctypes.data_as(_PLD),
                         off.ctypes.data_as(C.POINTER(C.c_long)))
    return dict(cos_theta=ct, sin_theta=st, nphi=nphi, phi0=ph, weight=w, offset=off)


def map_shape(sampling, L, nside=0):
    """MW [L, 2L-1]; MWSS [L+1, 2L]; DH [2L, 2L-1]; GL [L, 2L-1]; HEALPix [12 nside^2] (ring-ordered)."""
    if sampling == HEALPIX:
        return (12 * nside * nside,)
    return {MW: (L, 2 * L - 1), MWSS: (L + 1, 2 * L), DH: (2 * L, 2 * L - 1), GL: (L, 2 * L - 1)}[sampling]


# ---- S^2 ---------------------------------------------------------------------------------------------------
def s2_inverse(L, spin, sampling, flm, nside=0, direct=False):
    flm = _c128(flm, (L, 2 * L - 1))
    f = np.zeros(map_shape(sampling, L, nside), dtype=np.complex128)
    fn = lib().orc_s2_inverse_direct if direct else lib().orc_s2_inverse
    _check(fn(L, spin, sampling, nside, _pd(flm), _pd(f)), "s2_inverse")
    return f


def s2_forward(L, spin, sampling, f, nside=0, direct=False):
    f = _c128(f, map_shape(sampling, L, nside))
    flm = np.zeros((L, 2 * L - 1), dtype=np.complex128)
    fn = lib().orc_s2_forward_direct if direct else lib().orc_s2_forward
    _check(fn(L, spin, sampling, nside, _pd(f), _pd(flm)), "s2_forward")
    return flm


def s2_forward_iter(L, spin, sampling, f, niter, nside=0):
    """Forward transform with `niter` refinement iterations ("iterations are usually performed" on HEALPix; reading
    R24 of DESIGN.md): flm_0 = F f;  flm_{k+1} = flm_k + F (f - F^-1 flm_k).  A composition of the oracle's own F and F^-1."""
    f = _c128(f, map_shape(sampling, L, nside))
    flm = s2_forward(L, spin, sampling, f, nside)
    for _ in range(int(niter)):
        flm = flm + s2_forward(L, spin, sampling, f - s2_inverse(L, spin, sampling, flm, nside), nside)
    return flm


def s2_inverse_rings(L, spin, sampling, flm, rings, nside=0):
    """Samples of the selected rings only (list of 1-D complex arrays, one per ring)."""
    flm = _c128(flm, (L, 2 * L - 1))
    rings = np.ascontiguousarray(rings, dtype=np.int32)
    tab = ring_table(sampling, L, nside)
    lens = tab["nphi"][rings]
    out = np.zeros(int(lens.sum()), dtype=np.complex128)
    if len(rings) == 0:
        return []
    _check(lib().orc_s2_inverse_rings(L, spin, sampling, nside, _pd(flm), len(rings),
                                      rings.ctypes.data_as(_PI), _pd(out)), "s2_inverse_rings")
    return np.split(out, np.cumsum(lens)[:-1])


def s2_forward_columns(L, spin, sampling, f, ms, nside=0):
    """flm[:, m+L-1] for the selected m only: returns array [len(ms), L]."""
    f = _c128(f, map_shape(sampling, L, nside))
    ms = np.ascontiguousarray(ms, dtype=np.int32)
    out = np.zeros((len(ms), L), dtype=np.complex128)
    _check(lib().orc_s2_forward_columns(L, spin, sampling, nside, _pd(f), len(ms),
                                        ms.ctypes.data_as(_PI), _pd(out)), "s2_forward_columns")
    return out


def s2_theta_inverse_columns(L, spin, sampling, flm, ms, nside=0):
    """Eq. 33 only: F_m(theta_ring) for the selected m: returns array [len(ms), nrings]."""
    flm = _c128(flm, (L, 2 * L - 1))
    ms = np.ascontiguousarray(ms, dtype=np.int32)
    out = np.zeros((len(ms), num_rings(sampling, L, nside)), dtype=np.complex128)
    _check(lib().orc_s2_theta_inverse_columns(L, spin, sampling, nside, _pd(flm), len(ms),
                                              ms.ctypes.data_as(_PI), _pd(out)), "s2_theta_inverse_columns")
    return out


def s2_theta_forward_columns(L, spin, sampling, W, ms, nside=0):
    """Eq. 30 only: flm[:, m] = pref(l) sum_ring W[i, ring] d^l_{m,-s}(theta_ring) for the selected m (W already weighted);
    `sampling` may be any ring-set code incl. MW_QUAD / MWSS_QUAD.  Returns array [len(ms), L]."""
    ms = np.ascontiguousarray(ms, dtype=np.int32)
    W = _c128(W, (len(ms), num_rings(sampling, L, nside)))
    out = np.zeros((len(ms), L), dtype=np.complex128)
    _check(lib().orc_s2_theta_forward_columns(L, spin, sampling, nside, _pd(W), len(ms),
                                              ms.ctypes.data_as(_PI), _pd(out)), "s2_theta_forward_columns")
    return out


# ---- adjoints (Eq. 52 / 58): plain conjugate-transposed sums ------------------------------------------------
def s2_forward_adjoint(L, spin, sampling, flm, nside=0):
    """F^H: coefficients -> map, the conjugate transpose of s2_forward (Eq. 50-52)."""
    flm = _c128(flm, (L, 2 * L - 1))
    f = np.zeros(map_shape(sampling, L, nside), dtype=np.complex128)
    _check(lib().orc_s2_forward_adjoint(L, spin, sampling, nside, _pd(flm), _pd(f)), "s2_forward_adjoint")
    return f


def s2_inverse_adjoint_columns(L, spin, sampling, f, ms, nside=0):
    """(F^-1)^H for the selected m: returns array [len(ms), L] (Eq. 56-58)."""
    f = _c128(f, map_shape(sampling, L, nside))
    ms = np.ascontiguousarray(ms, dtype=np.int32)
    out = np.zeros((len(ms), L), dtype=np.complex128)
    _check(lib().orc_s2_inverse_adjoint_columns(L, spin, sampling, nside, _pd(f), len(ms),
                                                ms.ctypes.data_as(_PI), _pd(out)), "s2_inverse_adjoint_columns")
    return out


def s2_inverse_adjoint(L, spin, sampling, f, nside=0):
    """(F^-1)^H: map -> coefficients flm[L, 2L-1]."""
    ms = np.arange(-(L - 1), L)
    return np.ascontiguousarray(s2_inverse_adjoint_columns(L, spin, sampling, f, ms, nside).T)


# ---- SO(3) -------------------------------------------------------------------------------------------------
def so3_inverse(L, N, flmn):
    flmn = _c128(flmn, (2 * N - 1, L, 2 * L - 1))
    f = np.zeros((2 * N - 1, L, 2 * L - 1), dtype=np.complex128)
    _check(lib().orc_so3_inverse(L, N, _pd(flmn), _pd(f)), "so3_inverse")
    return f


def so3_forward(L, N, f):
    f = _c128(f, (2 * N - 1, L, 2 * L - 1))
    flmn = np.zeros((2 * N - 1, L, 2 * L - 1), dtype=np.complex128)
    _check(lib().orc_so3_forward(L, N, _pd(f), _pd(flmn)), "so3_forward")
    return flmn


# ---- SO(3) adjoints: the transposed chains of Eq. 15-18, step by step in reverse order ----
# The Wigner transform is, per order n of the gamma transform (Eq. 16), a spin transform with second index n (Eq. 15 / 18): with
# s = -n, W_n = (2 pi / (2N-1)) / p_s(l) * F_s and (W^-1)_n = F_s^-1 * ((2l+1)/(8 pi^2)) / p_s(l), p_s(l) = (-1)^s sqrt((2l+1)/(4 pi)) the
# prefactor of Eq. 30 / 33 (that relation is pinned in tests/test_oracle_so3.py).  The adjoints below transpose exactly that chain with
# the oracle's own (pinned) S^2 adjoints and plain gamma sums; they are pinned by the dot-product identity against so3_forward /
# so3_inverse (tests/test_oracle_adjoint.py).
def _so3_diag(L, n, num):
    l = np.arange(L, dtype=np.float64)
    p = (-1.0) ** n * np.sqrt((2 * l + 1) / (4 * np.pi))
    return (num(l) / p)[:, None]


def so3_forward_adjoint(L, N, flmn):
    """W^H: coefficients flmn[2N-1, L, 2L-1] -> f[2N-1 (gamma), L (beta), 2L-1 (alpha)], the conjugate transpose of so3_forward."""
    flmn = _c128(flmn, (2 * N - 1, L, 2 * L - 1))
    NG = 2 * N - 1
    g_n = np.zeros((NG, L, 2 * L - 1), dtype=np.complex128)
    for ni in range(NG):
        n = ni - (N - 1)
        y = flmn[ni] * _so3_diag(L, n, lambda l: np.full_like(l, 2 * np.pi / NG))       # transpose of the l-scaling (real, diagonal)
        g_n[ni] = s2_forward_adjoint(L, -n, 0, y)                                            # transpose of the spin transform with s = -n
    gam = 2 * np.pi * np.arange(NG) / NG
    ns = np.arange(NG) - (N - 1)
    # transpose of f_n = sum_g f e^{-i n gamma_g}:  f[g] = sum_n e^{+i n gamma_g} g_n
    return np.einsum("gn,nba->gba", np.exp(1j * np.outer(gam, ns)), g_n)


def so3_inverse_adjoint(L, N, f):
    """(W^-1)^H: f[2N-1, L, 2L-1] -> coefficients flmn[2N-1, L, 2L-1], the conjugate transpose of so3_inverse."""
    f = _c128(f, (2 * N - 1, L, 2 * L - 1))
    NG = 2 * N - 1
    gam = 2 * np.pi * np.arange(NG) / NG
    ns = np.arange(NG) - (N - 1)
    h_n = np.einsum("ng,gba->nba", np.exp(-1j * np.outer(ns, gam)), f)                       # transpose of f = sum_n e^{+i n gamma_g} (...)
    out = np.zeros((NG, L, 2 * L - 1), dtype=np.complex128)
    for ni in range(NG):
        n = ni - (N - 1)
        c = s2_inverse_adjoint(L, -n, 0, h_n[ni])
        out[ni] = c * _so3_diag(L, n, lambda l: (2 * l + 1) / (8 * np.pi ** 2))
    return out

"""Test-side helper: the projection the library applies to the theta = pi ring of an MW map (include/b200sht.h, s2_forward;
DESIGN.md R21), restated in numpy so that the ORACLE can be called on the projected array while the GPU gets the raw one.

A spin-s function has the single value c exp(i s phi) at theta = pi (only the order m = s survives, Eq. 29), so the
last ring of f[..., L, 2L-1] is replaced by its exp(i s phi) Fourier component; on SO(3), per order n of the gamma transform,
by its m = -n component (d^l_{mn}(pi) ~ delta_{m,-n})."""
import numpy as np


def project_mw_pole(f, spin):
    f = np.array(f, copy=True)
    ring = f[..., -1, :]
    n = ring.shape[-1]
    e = np.exp(2j * np.pi * spin * np.arange(n) / n)
    c = (ring * np.conj(e)).sum(-1, keepdims=True) / n
    out = c * e
    f[..., -1, :] = out.real if np.isrealobj(f) else out
    return f


def project_so3_pole(f):
    """f[2N-1, L, 2L-1] = (gamma, beta, alpha): project the beta = pi ring, for every gamma-order n, onto its m = -n alpha-order."""
    f = np.array(f, copy=True)
    ng, _, na = f.shape
    ring = f[:, -1, :]                                # [gamma, alpha]
    fn = np.fft.fft(ring, axis=0)                     # bins n mod (2N-1):  sum_g f e^{-i n gamma_g}
    a = np.arange(na)
    for b in range(ng):
        n = b if b <= ng // 2 else b - ng
        e = np.exp(-2j * np.pi * n * a / na)          # e^{i m alpha}, m = -n
        fn[b] = ((fn[b] * np.conj(e)).sum() / na) * e
    f[:, -1, :] = np.fft.ifft(fn, axis=0)
    return f


def project_mwss_poles(f, spin):
    """MWSS maps f[..., L+1, 2L] hold BOTH poles as rings: theta = 0 keeps only the order m = -s (Eq. 28), theta = pi only m = +s
    (Eq. 29)."""
    f = np.array(f, copy=True)
    n = f.shape[-1]
    p = np.arange(n)
    for ring, m in ((0, -spin), (-1, spin)):
        e = np.exp(2j * np.pi * m * p / n)
        c = (f[..., ring, :] * np.conj(e)).sum(-1, keepdims=True) / n
        out = c * e
        f[..., ring, :] = out.real if np.isrealobj(f) else out
    return f

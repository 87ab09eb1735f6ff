"""Seeded random sweep over the option space of S^2 plans: sampling x spin x reality x fold x symmetric-ring inverse x tile x paired theta-FFT
columns x CUDA graph, at band-limits that are not multiples of any tile size.  Every case: inverse against the oracle element by element,
forward of RAW white noise against the oracle (pole rings projected by the test, R21), exact-zero coefficients outside the support."""
import numpy as np
import pytest

from mwpole import project_mw_pole, project_mwss_poles
from paper_2311_14670_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
TOL = 1e-12


def rel(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


def cases(n=28, seed=20231114):
    rng = np.random.default_rng(seed)
    out = []
    for i in range(n):
        samp = ["mw", "mw", "mwss", "dh", "gl", "hp"][int(rng.integers(6))]
        L = int(rng.integers(2, 150))
        spin = int(rng.integers(-3, 4)) if rng.random() < 0.6 else 0
        if abs(spin) >= L:
            spin = 0
        real = bool(spin == 0 and rng.random() < 0.3)
        opt = lambda: [None, False, True][int(rng.integers(3))]
        kw = dict(fold=opt() if spin == 0 else None, invsym=opt(), tile=[None, 64, 128][int(rng.integers(3))], graph=opt())
        if samp in ("mw", "mwss"):
            kw["pair"] = opt()
        nside = int(2 ** rng.integers(0, 5)) if samp == "hp" else 0
        out.append(pytest.param(samp, L, spin, real, nside, kw, id=f"{i}-{samp}-L{L}-s{spin}{'-real' if real else ''}"))
    return out


@pytest.mark.parametrize("samp,L,spin,real,nside,kw", cases())
def test_random_plan_options_vs_oracle(orc, samp, L, spin, real, nside, kw):
    from paper_2311_14670_b200 import api
    gs, os_ = {"mw": (api.MW, orc.MW), "mwss": (api.MWSS, orc.MWSS), "dh": (api.DH, orc.DH), "gl": (api.GL, orc.GL), "hp": (api.HEALPIX, orc.HEALPIX)}[samp]
    P = api.Plan(L, spin, sampling=gs, nside=nside, reality=real, **kw)
    okw = dict(nside=nside) if samp == "hp" else {}
    flm = synth.random_flm(L, spin, seed=100 + L + 11 * spin, real=real)
    ref = orc.s2_inverse(L, spin, os_, flm, **okw)
    got = P.inverse(torch.from_numpy(flm).cuda()).cpu().numpy()
    assert rel(got, ref.real if real else ref) < TOL
    shape = (12 * nside * nside,) if samp == "hp" else orc.map_shape(os_, L)
    g = synth.random_map(shape, seed=100 + 3 * L + spin, real=real)
    gp = project_mw_pole(g, spin) if samp == "mw" else project_mwss_poles(g, spin) if samp == "mwss" else g
    want = orc.s2_forward(L, spin, os_, gp.astype(np.complex128), **okw)
    back = P.forward(torch.from_numpy(g).cuda()).cpu().numpy()
    assert rel(back, want) < TOL
    el = np.arange(L)[:, None]
    m = np.arange(-(L - 1), L)[None, :]
    assert np.all(back[(np.abs(m) > el) | (el < abs(spin))] == 0)
    # a second call on the same buffers (graph replay where the plan uses graphs) gives the same numbers
    again = P.forward(torch.from_numpy(g).cuda()).cpu().numpy()
    assert rel(again, back) < 1e-13

"""The test-side pole-ring projection (tests/mwpole.py) must be the identity on samples of genuine spin-s functions -- that is what
makes "oracle(project(raw))" the right expectation for the library's forward transform of raw arrays (R21)."""
import numpy as np
import pytest

from mwpole import project_mw_pole, project_so3_pole
from paper_2311_14670_b200 import synth


@pytest.mark.parametrize("spin", [0, 1, -2, 3])
def test_projection_is_identity_on_band_limited_maps(orc, spin):
    L = 9
    f = orc.s2_inverse(L, spin, orc.MW, synth.random_flm(L, spin, seed=spin + 5))
    assert np.abs(project_mw_pole(f, spin) - f).max() < 1e-14 * np.abs(f).max()
    g = synth.random_map((L, 2 * L - 1), seed=1)
    p = project_mw_pole(g, spin)
    assert np.array_equal(p[:-1], g[:-1]) and np.abs(project_mw_pole(p, spin) - p).max() < 1e-15      # idempotent, other rings untouched
    assert np.abs(p[-1] - g[-1]).max() > 0.1                                                          # ... and it does change raw noise


def test_so3_projection_is_identity_on_band_limited_functions(orc):
    L, N = 7, 3
    f = orc.so3_inverse(L, N, synth.random_flmn(L, N, seed=2))
    assert np.abs(project_so3_pole(f) - f).max() < 1e-14 * np.abs(f).max()
    g = synth.random_map((2 * N - 1, L, 2 * L - 1), seed=4)
    p = project_so3_pole(g)
    assert np.abs(project_so3_pole(p) - p).max() < 1e-14 and np.array_equal(p[:, :-1], g[:, :-1])


def test_real_maps_keep_the_ring_mean(orc):
    g = synth.random_map((6, 11), seed=3, real=True)
    p = project_mw_pole(g, 0)
    assert p.dtype == np.float64 and np.allclose(p[-1], g[-1].mean())

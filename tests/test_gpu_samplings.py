"""GPU parity of the MWSS, DH and Gauss-Legendre samplings against the CPU oracle, element by
element: inverse, forward of the oracle's map (= the generating coefficients, sampling theorem), forward of RAW white noise
(MWSS: against the oracle on the array whose two pole rings are projected, R21), folds forced both ways, real maps,
plus one sampled comparison per sampling at L = 2048."""
import numpy as np
import pytest

from mwpole import project_mwss_poles
from paper_2311_14670_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
TOL = 1e-12


def rel(a, b, scale=None):
    return float(np.abs(a - b).max() / (np.abs(b).max() if scale is None else scale))


@pytest.fixture(scope="module")
def api():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2311_14670_b200 import api as A
    return A


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def codes(api, orc, name):
    return {"mwss": (api.MWSS, orc.MWSS), "dh": (api.DH, orc.DH), "gl": (api.GL, orc.GL)}[name]


@pytest.mark.parametrize("name", ["mwss", "dh", "gl"])
@pytest.mark.parametrize("L,spin", [(1, 0), (2, 0), (3, 1), (8, 0), (33, 0), (64, 2), (48, -3), (130, 1), (131, -2), (200, 0), (257, 2)])
def test_inverse_and_forward_vs_oracle(api, orc, name, L, spin):
    gs, os_ = codes(api, orc, name)
    flm = synth.random_flm(L, spin, seed=L + 7 * spin)
    P = api.Plan(L, spin, sampling=gs)
    assert P.map_shape == orc.map_shape(os_, L)
    f = P.inverse(dev(flm)).cpu().numpy()
    f_ref = orc.s2_inverse(L, spin, os_, flm)
    assert rel(f, f_ref) < TOL
    back = P.forward(dev(f_ref)).cpu().numpy()
    assert rel(back, orc.s2_forward(L, spin, os_, f_ref)) < TOL
    assert rel(back, flm) < TOL                                  # sampling theorem: exact round trip
    el = np.arange(L)[:, None]
    m = np.arange(-(L - 1), L)[None, :]
    assert np.all(back[(np.abs(m) > el) | (el < abs(spin))] == 0)


@pytest.mark.parametrize("name", ["mwss", "dh", "gl"])
@pytest.mark.parametrize("fold", [False, True])
@pytest.mark.parametrize("L,spin,real", [(9, 0, False), (40, 0, False), (40, 1, False), (65, -2, False), (130, 0, True), (96, 0, False)])
def test_forward_of_raw_white_noise_and_folds(api, orc, name, fold, L, spin, real):
    """Forward of a RAW white-noise map (not band-limited) with the north-south fold of spin-0 plans forced off / on; the inverse of
    the same plan runs folded / unfolded accordingly.  MWSS: the oracle gets the array with both pole rings projected (R21)."""
    gs, os_ = codes(api, orc, name)
    g = synth.random_map(orc.map_shape(os_, L), seed=3 * L + spin, real=real)
    P = api.Plan(L, spin, sampling=gs, reality=real, fold=fold)
    got = P.forward(dev(g)).cpu().numpy()
    gp = project_mwss_poles(g, spin) if name == "mwss" else g
    assert rel(got, orc.s2_forward(L, spin, os_, gp.astype(np.complex128))) < TOL
    flm = synth.random_flm(L, spin, seed=5 * L, real=real)
    ref = orc.s2_inverse(L, spin, os_, flm)
    f = P.inverse(dev(flm)).cpu().numpy()
    assert rel(f, ref.real if real else ref) < TOL
    if name == "mwss":
        raw = orc.s2_forward(L, spin, os_, g.astype(np.complex128))
        print(f"MWSS L={L} spin={spin}: departure from the oracle on the raw array {rel(got, raw):.3e}")


@pytest.mark.parametrize("L,spin", [(2, 0), (9, 0), (40, 1), (65, -2), (128, 0)])
def test_mwss_forward_with_one_order_per_theta_fft_column(api, orc, L, spin):
    """MWSS forward with SHT_OPT_NO_PAIR (the default carries two orders per theta-FFT column, tested above) on raw white noise."""
    g = synth.random_map(orc.map_shape(orc.MWSS, L), seed=7 * L + spin)
    P = api.Plan(L, spin, sampling=api.MWSS, pair=False)
    want = orc.s2_forward(L, spin, orc.MWSS, project_mwss_poles(g, spin).astype(np.complex128))
    assert rel(P.forward(dev(g)).cpu().numpy(), want) < TOL


@pytest.mark.parametrize("name", ["mwss", "dh", "gl"])
def test_theta_stage_entry_points(api, orc, name):
    """Hot path alone on the new ring sets: Eq. 33 against the oracle's F_m(theta) columns (pole rings included)."""
    gs, os_ = codes(api, orc, name)
    L, spin = 72, 2
    flm = synth.random_flm(L, spin, seed=4)
    P = api.Plan(L, spin, sampling=gs)
    F = P.theta_inverse(dev(flm)).cpu().numpy()
    ms = np.arange(-(L - 1), L)
    assert F.shape[1] == orc.num_rings(os_, L)
    assert rel(F, orc.s2_theta_inverse_columns(L, spin, os_, flm, ms)) < TOL


@pytest.mark.parametrize("name", ["mwss", "dh", "gl"])
def test_L2048_sampled(api, orc, name):
    """One sampled comparison per sampling at the size the north_star target is stated on (L = 2048, spin 0): a few rings of the
    inverse (poles, first ring, equator), a few orders m of the forward of a raw white-noise map, and the exact round trip."""
    gs, os_ = codes(api, orc, name)
    L = 2048
    flm = synth.random_flm(L, 0, seed=4, sigma=synth.SIGMA_RED)
    P = api.Plan(L, 0, sampling=gs)
    d = dev(flm)
    f = P.inverse(d)
    back = P.forward(f)
    assert float((back - d).abs().max() / d.abs().max()) < 1e-11
    nr = orc.num_rings(os_, L)
    rings = np.array([0, 1, nr // 2, nr - 2, nr - 1])
    rows = orc.s2_inverse_rings(L, 0, os_, flm, rings)
    scale = max(np.abs(r).max() for r in rows)
    fh = f.cpu().numpy()
    for r, row in zip(rings, rows):
        assert rel(fh[r], row, scale) < 1e-11, r
    g = synth.random_map(orc.map_shape(os_, L), seed=31)
    got = P.forward(dev(g)).cpu().numpy()
    ms = np.array([-(L - 1), -1, 0, 1, 2, 1024, L - 1])
    gp = project_mwss_poles(g, 0) if name == "mwss" else g
    want = orc.s2_forward_columns(L, 0, os_, gp, ms)
    sc = np.abs(want).max()
    for m, col in zip(ms, want):
        assert rel(got[:, m + L - 1], col, sc) < 1e-11, m

"""GPU parity of the adjoint entry points (Sec. 5.3-5.4): the dot-product identities
<F x, y> = <x, F^H y>, <F^-1 c, g> = <c, (F^-1)^H g> on random (not band-limited) vectors, element-wise parity against the CPU
oracle's adjoints (plain conjugate-transposed sums), Eq. 52 on a direct-quadrature sampling, and the theta-step-only forms
(Eq. 63 / 68) against the theta-stage entry points they transpose."""
import numpy as np
import pytest

from mwpole import project_mw_pole, project_mwss_poles
from paper_2311_14670_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
TOL = 1e-12


def rel(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


@pytest.fixture(scope="module")
def api():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2311_14670_b200 import api as A
    return A


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def plan_for(api, orc, name, L, spin, **kw):
    nside = kw.pop("nside", 0)
    gs, os_ = {"mw": (api.MW, orc.MW), "mwss": (api.MWSS, orc.MWSS), "dh": (api.DH, orc.DH), "gl": (api.GL, orc.GL),
               "hp": (api.HEALPIX, orc.HEALPIX)}[name]
    return api.Plan(L, spin, sampling=gs, nside=nside, adjoint=True, **kw), os_


CASES = [("mw", 0), ("mwss", 0), ("dh", 0), ("gl", 0), ("hp", 8)]


@pytest.mark.parametrize("name,nside", CASES)
@pytest.mark.parametrize("L,spin", [(8, 0), (33, 0), (40, 2), (64, -1), (130, 2), (200, 0), (257, 2), (1030, 1)])     # (1030: transforms start from the silent-head state)
def test_dot_product_identities(api, orc, name, nside, L, spin):
    P, os_ = plan_for(api, orc, name, L, spin, nside=nside)
    x = synth.random_map(P.map_shape, seed=L)
    y = synth.random_flm(L, spin, seed=L + 1)
    Fx = P.forward(dev(x)).cpu().numpy()
    FHy = P.forward_adjoint(dev(y)).cpu().numpy()
    a, b = np.vdot(y, Fx), np.vdot(FHy, x)
    assert abs(a - b) < TOL * abs(a), (a, b)
    c = synth.random_flm(L, spin, seed=L + 2)
    g = synth.random_map(P.map_shape, seed=L + 3)
    Ic = P.inverse(dev(c)).cpu().numpy()
    IHg = P.inverse_adjoint(dev(g)).cpu().numpy()
    a, b = np.vdot(g, Ic), np.vdot(IHg, c)
    assert abs(a - b) < TOL * abs(a), (a, b)
    el = np.arange(L)[:, None]
    m = np.arange(-(L - 1), L)[None, :]
    assert np.all(IHg[(np.abs(m) > el) | (el < abs(spin))] == 0)


@pytest.mark.parametrize("name,nside", CASES)
@pytest.mark.parametrize("L,spin", [(12, 0), (33, 2), (64, 0), (96, -2)])
def test_adjoints_vs_oracle(api, orc, name, nside, L, spin):
    """Element by element against the oracle's conjugate-transposed sums.  MW / MWSS: the library's forward transform projects the
    pole ring(s) (R21), F_gpu = F_oracle P, so its adjoint is P F_oracle^H: the same projection applied to the output."""
    P, os_ = plan_for(api, orc, name, L, spin, nside=nside)
    y = synth.random_flm(L, spin, seed=7 * L)
    got = P.forward_adjoint(dev(y)).cpu().numpy()
    want = orc.s2_forward_adjoint(L, spin, os_, y, nside=nside)
    if name == "mw":
        want = project_mw_pole(want, spin)
    if name == "mwss":
        want = project_mwss_poles(want, spin)
    assert rel(got, want) < TOL
    g = synth.random_map(P.map_shape, seed=9 * L)
    got = P.inverse_adjoint(dev(g)).cpu().numpy()
    assert rel(got, orc.s2_inverse_adjoint(L, spin, os_, g, nside=nside)) < TOL


@pytest.mark.parametrize("name,nside", CASES)
def test_theta_step_adjoints(api, orc, name, nside):
    """Eq. 63 / 68: the theta-step-only forms are the conjugate transposes of the theta-stage entry points."""
    L, spin = 72, 2
    P, os_ = plan_for(api, orc, name, L, spin, nside=nside)
    rng = np.random.default_rng(5)
    nq, nt = P.ntheta(True), P.ntheta(False)
    W = rng.standard_normal((2 * L - 1, nq)) + 1j * rng.standard_normal((2 * L - 1, nq))
    y = synth.random_flm(L, spin, seed=3)
    a = np.vdot(y, P.theta_forward(dev(W)).cpu().numpy())
    b = np.vdot(P.theta_forward_adjoint(dev(y)).cpu().numpy(), W)
    assert abs(a - b) < TOL * abs(a)
    Fm = rng.standard_normal((2 * L - 1, nt)) + 1j * rng.standard_normal((2 * L - 1, nt))
    c = synth.random_flm(L, spin, seed=4)
    a = np.vdot(Fm, P.theta_inverse(dev(c)).cpu().numpy())
    b = np.vdot(P.theta_inverse_adjoint(dev(Fm)).cpu().numpy(), c)
    assert abs(a - b) < TOL * abs(a)
    # Eq. 67: (F_Theta^-1)^H is the unweighted analysis sum -- against the oracle's theta-forward columns on the map's rings
    ms = np.arange(-(L - 1), L)
    want = orc.s2_theta_forward_columns(L, spin, os_, Fm, ms, nside=nside).T
    assert rel(P.theta_inverse_adjoint(dev(Fm)).cpu().numpy(), want) < TOL


def test_eq52_on_dh_and_errors_without_the_option(api, orc):
    L, spin = 48, 1
    P, os_ = plan_for(api, orc, "dh", L, spin)
    y = synth.random_flm(L, spin, seed=2)
    tab = orc.ring_table(os_, L)
    q = np.asarray(tab["weight"], float)[:, None]
    lhs = P.forward_adjoint(dev(y)).cpu().numpy()
    rhs = q * P.inverse(dev(y)).cpu().numpy()                       # F^H = Q F^-1
    assert rel(lhs, rhs) < TOL
    from paper_2311_14670_b200._lib import ShtError
    P0 = api.Plan(L, spin)
    with pytest.raises(ShtError):
        P0.forward_adjoint(dev(y))
    with pytest.raises(ShtError):
        api.Plan(L, 0, reality=True, adjoint=True)


@pytest.mark.parametrize("L,N", [(6, 3), (24, 4), (40, 8), (65, 5)])
def test_so3_adjoints_dot_products_and_oracle(api, orc, L, N):
    """Wigner adjoints (so3_forward_adjoint_plan / so3_inverse_adjoint_plan): <W x, y> = <x, W^H y> and <W^-1 c, g> = <c, W^-H g> on random
    arrays against the library's own transforms, and element-wise parity with the oracle's transposed chains (the library's forward is
    W_oracle P with the pole-ring projection P of R21, so its adjoint is P W_oracle^H: the test applies P to the oracle's output)."""
    from mwpole import project_so3_pole
    shape = (2 * N - 1, L, 2 * L - 1)
    P = api.Plan(L, N=N, adjoint=True)
    x = synth.random_map(shape, seed=1); y = synth.random_flmn(L, N, seed=2)
    c = synth.random_flmn(L, N, seed=3); g = synth.random_map(shape, seed=4)
    Wx = P.forward(dev(x)).cpu().numpy()
    WHy = P.forward_adjoint(dev(y)).cpu().numpy()
    a, b = np.vdot(y, Wx), np.vdot(WHy, x)
    assert abs(a - b) < 1e-12 * abs(a)
    Vc = P.inverse(dev(c)).cpu().numpy()
    VHg = P.inverse_adjoint(dev(g)).cpu().numpy()
    a, b = np.vdot(g, Vc), np.vdot(VHg, c)
    assert abs(a - b) < 1e-12 * abs(a)
    if L <= 40:
        assert rel(WHy, project_so3_pole(orc.so3_forward_adjoint(L, N, y))) < TOL
        assert rel(VHg, orc.so3_inverse_adjoint(L, N, g)) < TOL
    with pytest.raises(Exception):
        api.Plan(8, N=2).forward_adjoint(dev(synth.random_flmn(8, 2, seed=1)))       # plan without SHT_OPT_ADJOINT

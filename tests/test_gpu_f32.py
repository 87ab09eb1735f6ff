"""GPU parity of the fp32 variant (BASELINE.json configs[4]: "fp64 and fp32"): spin-0 MW plans whose fused recursion +
contraction kernels compute in fp32 (csrc/theta_f32.cu).  Tolerance from north_star: max|delta| / max|ref| <= 1e-4, both sides
deciding nothing in floating point (linear maps), against the fp64/long-double CPU oracle on the same seeded inputs."""
import numpy as np
import pytest

from paper_2311_14670_b200 import synth
from mwpole import project_mw_pole

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
TOL32 = 1e-4


def rel(a, b, scale=None):
    return float(np.abs(a - b).max() / (np.abs(b).max() if scale is None else scale))


@pytest.fixture(scope="module")
def api():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2311_14670_b200 import api as A
    return A


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("L,real", [(1, False), (2, False), (8, False), (33, False), (64, False), (130, False), (200, True), (257, False), (512, False)])
def test_f32_inverse_forward_vs_oracle(api, orc, L, real):
    flm = synth.random_flm(L, 0, seed=11 * L, sigma=synth.SIGMA_RED, real=real)
    P = api.Plan(L, 0, reality=real, dtype="f32")
    f = P.inverse(dev(flm.astype(np.complex64))).cpu().numpy()
    assert f.dtype == (np.float32 if real else np.complex64)
    f_ref = orc.s2_inverse(L, 0, orc.MW, flm)
    f_ref = f_ref.real if real else f_ref
    assert rel(f, f_ref) < TOL32
    back = P.forward(dev(f_ref.astype(f.dtype))).cpu().numpy()
    assert back.dtype == np.complex64
    assert rel(back, flm) < TOL32                                 # sampling theorem (pin 6), at fp32 accuracy
    g = synth.random_map((L, 2 * L - 1), seed=L, real=real)
    got = P.forward(dev(g.astype(f.dtype))).cpu().numpy()
    assert rel(got, orc.s2_forward(L, 0, orc.MW, project_mw_pole(g, 0).astype(np.complex128))) < TOL32
    el = np.arange(L)[:, None]
    m = np.arange(-(L - 1), L)[None, :]
    assert np.all(back[np.abs(m) > el] == 0)


def test_f32_unsupported_requests_are_refused(api):
    from paper_2311_14670_b200._lib import ShtError
    # (a batch is accepted: it runs map by map; every sampling and every spin is served)
    for kw in (dict(N=3, adjoint=True), dict(spin=2, adjoint=True), dict(spin=0, adjoint=True), dict(spin=0, precompute=True), dict(spin=1, precompute=True)):
        with pytest.raises(ShtError):
            api.Plan(16, dtype="f32", **kw)
    P = api.Plan(16, 2, dtype="f32")
    with pytest.raises(ShtError):                # the theta-stage entry points take fp64 arrays: fp64 plans only
        P.theta_inverse(torch.zeros((16, 31), dtype=torch.complex128, device="cuda"))


@pytest.mark.parametrize("L,spin,sampling", [(33, 1, "mw"), (130, -2, "mw"), (257, 2, "mw"), (64, 2, "dh"), (48, -1, "mwss"), (40, 2, "gl")])
def test_f32_arrays_with_spin_run_the_fp64_kernels(api, orc, L, spin, sampling):
    """SHT_F32 with spin != 0: fp32 public arrays around the fp64 kernels (the fp32 kernels recurse n = 0 only).  The result is the fp64
    transform of the fp32-rounded input, rounded to fp32: well inside the fp32 tolerance, asserted at 2e-6."""
    code = {"mw": api.MW, "dh": api.DH, "mwss": api.MWSS, "gl": api.GL}[sampling]
    oc = {"mw": orc.MW, "dh": orc.DH, "mwss": orc.MWSS, "gl": orc.GL}[sampling]
    flm = synth.random_flm(L, spin, seed=3 * L + spin, sigma=synth.SIGMA_RED)
    P = api.Plan(L, spin, sampling=code, dtype="f32")
    f = P.inverse(dev(flm.astype(np.complex64))).cpu().numpy()
    assert f.dtype == np.complex64 and f.shape == tuple(P.map_shape)
    f_ref = orc.s2_inverse(L, spin, oc, flm)
    assert rel(f, f_ref) < 2e-6
    back = P.forward(dev(f_ref.astype(np.complex64))).cpu().numpy()
    assert back.dtype == np.complex64
    assert rel(back, flm) < 2e-6
    P64 = api.Plan(L, spin, sampling=code)
    f64 = P64.inverse(dev(flm.astype(np.complex64).astype(np.complex128))).cpu().numpy()
    assert np.array_equal(f, f64.astype(np.complex64)) or rel(f, f64) < 1e-7      # same kernels, rounded once on the way out


def test_f32_config5a_scale_L2048_sampled(api, orc):
    """fp32 at a size with deep underflow of the start values (2^-9000 at the first rings): sampled rings / orders vs the oracle."""
    L = 2048
    flm = synth.random_flm(L, 0, seed=4, sigma=synth.SIGMA_RED)
    P = api.Plan(L, 0, dtype="f32")
    f = P.inverse(dev(flm.astype(np.complex64))).cpu().numpy()
    rings = np.array([0, 1, 2, 1000, 2046, 2047])
    rows = orc.s2_inverse_rings(L, 0, orc.MW, flm, rings)
    scale = max(np.abs(r).max() for r in rows)
    for r, row in zip(rings, rows):
        assert rel(f[r], row, scale) < TOL32, r
    back = P.forward(dev(f)).cpu().numpy()
    assert rel(back, flm) < 2 * TOL32                             # two fp32 transforms in a row
    g = synth.random_map((L, 2 * L - 1), seed=15)
    got = P.forward(dev(g.astype(np.complex64))).cpu().numpy()
    ms = np.array([-(L - 1), -1, 0, 1, 2, 1024, L - 1])
    want = orc.s2_forward_columns(L, 0, orc.MW, project_mw_pole(g, 0), ms)
    sc = np.abs(want).max()
    for m, col in zip(ms, want):
        assert rel(got[:, m + L - 1], col, sc) < TOL32, m


@pytest.mark.parametrize("L,real", [(8, False), (33, False), (130, False), (200, True)])
def test_f32_forward_with_north_south_fold(api, orc, L, real):
    """fp32 forward with the north-south fold forced on (default at L >= 2048): northern rings only, E / O operand sets."""
    g = synth.random_map((L, 2 * L - 1), seed=3 * L, real=real)
    P = api.Plan(L, 0, reality=real, dtype="f32", fold=True)
    got = P.forward(dev(g.astype(np.float32 if real else np.complex64))).cpu().numpy()
    assert rel(got, orc.s2_forward(L, 0, orc.MW, project_mw_pole(g, 0).astype(np.complex128))) < TOL32


@pytest.mark.parametrize("name,nside,real", [("mwss", 0, False), ("dh", 0, False), ("gl", 0, True), ("hp", 16, True), ("hp", 32, False)])
@pytest.mark.parametrize("L,fold", [(40, None), (130, True), (130, False)])
def test_f32_other_samplings_vs_oracle(api, orc, name, nside, real, L, fold):
    """The fp32 kernels recurse the second index n = 0 on any ring set: spin-0 plans of every sampling, folded or not, within 1e-4 of the
    oracle (inverse, and forward of the oracle's map)."""
    gs, os_ = {"mwss": (api.MWSS, orc.MWSS), "dh": (api.DH, orc.DH), "gl": (api.GL, orc.GL), "hp": (api.HEALPIX, orc.HEALPIX)}[name]
    okw = dict(nside=nside) if name == "hp" else {}
    P = api.Plan(L, 0, sampling=gs, nside=nside, reality=real, dtype="f32", fold=fold)
    flm = synth.random_flm(L, 0, seed=7 + L, sigma=synth.SIGMA_RED, real=real)
    ref = orc.s2_inverse(L, 0, os_, flm, **okw)
    ref = ref.real if real else ref
    got = P.inverse(torch.from_numpy(flm.astype(np.complex64)).cuda()).cpu().numpy()
    assert float(np.abs(got - ref).max() / np.abs(ref).max()) < 1e-4
    want = orc.s2_forward(L, 0, os_, ref.astype(np.complex128), **okw)
    back = P.forward(torch.from_numpy(ref.astype(np.float32 if real else np.complex64)).cuda()).cpu().numpy()
    assert float(np.abs(back - want).max() / np.abs(want).max()) < 1e-4


@pytest.mark.parametrize("L,N", [(16, 3), (40, 8), (130, 2)])
def test_f32_arrays_so3_run_the_fp64_kernels(api, orc, L, N):
    """sht_plan_so3 with SHT_F32: complex64 arrays around the fp64 kernels (Eq. 15-18 need the orders n != 0)."""
    flmn = synth.random_flmn(L, N, seed=L + N)
    P = api.Plan(L, N=N, dtype="f32")
    f = P.inverse(dev(flmn.astype(np.complex64))).cpu().numpy()
    assert f.dtype == np.complex64 and f.shape == (2 * N - 1, L, 2 * L - 1)
    f_ref = orc.so3_inverse(L, N, flmn)
    assert rel(f, f_ref) < 2e-6
    back = P.forward(dev(f_ref.astype(np.complex64))).cpu().numpy()
    assert back.dtype == np.complex64 and rel(back, flmn) < 2e-6


@pytest.mark.parametrize("spin,real,tol", [(0, False, 1e-4), (0, True, 1e-4), (2, False, 2e-6)])
def test_f32_healpix_refinement_keeps_fp64_state(api, spin, real, tol):
    """s2_forward_iter_plan on a plan with fp32 arrays: the running coefficients and the residual stay in fp64 between the transforms, so the
    result follows the fp64 plan's iteration on the same (fp32-rounded) map."""
    nside, L, niter = 16, 32, 3
    rng = np.random.default_rng(7 + spin)
    g = rng.standard_normal(12 * nside * nside) + (0 if real else 1j * rng.standard_normal(12 * nside * nside))
    g32 = g.astype(np.float32 if real else np.complex64)
    P32 = api.Plan(L, spin, sampling=api.HEALPIX, nside=nside, reality=real, dtype="f32")
    P64 = api.Plan(L, spin, sampling=api.HEALPIX, nside=nside, reality=real)
    want = P64.forward_iter(dev(g32.astype(np.float64 if real else np.complex128)), niter).cpu().numpy()
    got = P32.forward_iter(dev(g32), niter).cpu().numpy()
    assert got.dtype == np.complex64
    assert rel(got, want) < tol
    zero = P32.forward_iter(dev(g32), 0).cpu().numpy()
    assert rel(zero, P32.forward(dev(g32)).cpu().numpy()) < 1e-6       # niter = 0 is the forward transform


def test_f32_arrays_with_spin_at_a_size_with_the_silent_head_skip(api, orc):
    """fp32 arrays around the fp64 kernels at L >= 1024, where the fp64 kernels start from the stored silent-head state: sampled rings and a
    round trip."""
    L, spin = 1030, 1
    flm = synth.random_flm(L, spin, seed=21, sigma=synth.SIGMA_RED)
    P = api.Plan(L, spin, dtype="f32")
    f = P.inverse(dev(flm.astype(np.complex64))).cpu().numpy()
    rings = np.array([0, 1, 7, 500, 1028, 1029])
    rows = orc.s2_inverse_rings(L, spin, orc.MW, flm, rings)
    scale = max(np.abs(r).max() for r in rows)
    for r, row in zip(rings, rows):
        assert rel(f[r], row, scale) < 2e-6, r
    back = P.forward(dev(f)).cpu().numpy()
    assert rel(back, flm) < 2e-6

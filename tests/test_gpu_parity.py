"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on seeded inputs.

Tolerance: fp64 max|delta| / max|ref| <= 1e-11 (BASELINE.json north_star) -- asserted here at 1e-12 for L <= 256,
which is still > 50x the errors observed (~3.5e-16 L)."""
import os

import numpy as np
import pytest

from paper_2311_14670_b200 import synth
from mwpole import project_mw_pole, project_so3_pole

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
TOL = 1e-12
HERE = os.path.dirname(os.path.abspath(__file__))


def rel(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


@pytest.fixture(scope="module")
def api():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2311_14670_b200 import api as A
    return A


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# sizes span several kernel tiles (128 degrees / 32 rings inverse; 32 degrees / 128 rings forward) plus ragged tails
@pytest.mark.parametrize("L,spin", [(1, 0), (2, 0), (3, 1), (8, 0), (33, 0), (64, 0), (64, 2), (48, -3), (130, 1), (131, -2), (200, 0), (257, 2)])
def test_s2_mw_inverse_forward_vs_oracle(api, orc, L, spin):
    flm = synth.random_flm(L, spin, seed=L + 7 * spin)
    P = api.Plan(L, spin)
    f = P.inverse(dev(flm)).cpu().numpy()
    f_ref = orc.s2_inverse(L, spin, orc.MW, flm)
    assert rel(f, f_ref) < TOL
    # forward of the oracle's map, against the oracle's forward AND against the generating coefficients (pin 6)
    back = P.forward(dev(f_ref)).cpu().numpy()
    assert rel(back, orc.s2_forward(L, spin, orc.MW, f_ref)) < TOL
    assert rel(back, flm) < TOL
    # coefficients outside the support are written as exact zeros
    el = np.arange(L)[:, None]
    m = np.arange(-(L - 1), L)[None, :]
    assert np.all(back[(np.abs(m) > el) | (el < abs(spin))] == 0)


def test_config1_L64_spin0_round_trip_and_forward(api, orc):
    """BASELINE.json configs[0]: spin-0 complex, MW L=64, flm iid complex N(0,1), seed 0."""
    L = 64
    flm = synth.random_flm(L, 0, seed=0)
    d = dev(flm)
    f = api.s2_inverse(d, L, 0)
    back = api.s2_forward(f, L, 0)
    assert rel(f.cpu().numpy(), orc.s2_inverse(L, 0, orc.MW, flm)) < TOL
    assert rel(back.cpu().numpy(), flm) < TOL
    # Table 1 of the paper: 1.2e-15 at L=64 (norm unspecified): same order of magnitude or better
    tab = {}
    for line in open(os.path.join(HERE, "golden", "paper_tables_roundtrip.txt")):
        if line.startswith("sht"):
            _, l_, e_ = line.split(); tab[int(l_)] = float(e_)
    sup = flm != 0
    assert np.abs(back.cpu().numpy() - flm)[sup].mean() < 10 * tab[64]


@pytest.mark.parametrize("L,spin", [(40, 1), (33, 0), (64, -2), (130, 2)])
def test_forward_of_raw_white_noise_matches_oracle_on_projected_pole_ring(api, orc, L, spin):
    """The forward transform is defined by the algorithm (upsampling + quadrature) for any array, not just band-limited maps.
    The GPU gets RAW white noise; the library projects the theta = pi ring onto exp(i s phi) (include/b200sht.h, R21), so
    the oracle is called on the array with that projection applied by the test.  The size of the departure from the paper's
    MW(2L)-grid algorithm on the raw array (which is ring-set dependent there) is measured and printed, not hidden."""
    f = synth.random_map((L, 2 * L - 1), seed=9 + L)
    P = api.Plan(L, spin)
    got = P.forward(dev(f)).cpu().numpy()
    fp = project_mw_pole(f, spin)
    assert rel(got, orc.s2_forward(L, spin, orc.MW, fp)) < TOL
    assert rel(P.forward(dev(fp)).cpu().numpy(), got) < 1e-14          # the projection is idempotent inside the library
    raw = orc.s2_forward(L, spin, orc.MW, f)
    dep = rel(got, raw)
    print(f"L={L} spin={spin}: max|GPU(raw) - oracle(raw)| / max|oracle(raw)| = {dep:.3e} (white noise on the pole ring; "
          f"pole-ring rms {np.abs(f[-1]).std():.2f})")
    # the departure is confined to the odd-symmetry component of the single pole ring: one ring of L, weight ~ 1/L^2
    assert dep < 0.5


def test_so3_forward_of_raw_white_noise(api, orc):
    L, N = 24, 4
    g = synth.random_map((2 * N - 1, L, 2 * L - 1), seed=77)
    P = api.Plan(L, N=N)
    got = P.forward(dev(g)).cpu().numpy()
    assert rel(got, orc.so3_forward(L, N, project_so3_pole(g))) < TOL
    print(f"SO(3) L={L} N={N}: departure from the oracle on the raw array {rel(got, orc.so3_forward(L, N, g)):.3e}")


def test_theta_stage_entry_points(api, orc):
    """Hot path alone: F_m(theta) of Eq. 33 against the oracle's columns; Eq. 30 on weighted rows."""
    L, spin = 96, 2
    flm = synth.random_flm(L, spin, seed=4)
    P = api.Plan(L, spin)
    F = P.theta_inverse(dev(flm)).cpu().numpy()
    ms = np.arange(-(L - 1), L)
    assert rel(F, orc.s2_theta_inverse_columns(L, spin, orc.MW, flm, ms)) < TOL
    # forward theta step (Eq. 30) on arbitrary weighted rows W[m][u], u indexing the library's quadrature rings
    # theta'_u = (2u+1) pi / (4L) (include/b200sht.h), against a direct sum with the oracle's d-functions
    nq = P.ntheta(True)
    assert nq == 2 * L
    rng = np.random.default_rng(0)
    W = (rng.standard_normal((2 * L - 1, nq)) + 1j * rng.standard_normal((2 * L - 1, nq)))
    out = P.theta_forward(dev(W)).cpu().numpy()
    # out[l, m] = pref(l) * sum_u W[m, u] d^l_{m,-s}(theta'_u)
    el = np.arange(L)
    pref = (-1.0) ** spin * np.sqrt((2 * el + 1) / (4 * np.pi))
    half = np.pi * (2 * np.arange(nq) + 1) / (8 * L)
    for m in (-(L - 1), -5, 0, 2, 31, L - 1):
        acc = np.zeros(L, complex)
        for u in range(nq):
            d = np.asarray(orc.d_lrec(L, m, -spin, cos_half=np.cos(half[u]), sin_half=np.sin(half[u])), float)
            acc += W[m + L - 1, u] * d
        want = pref * acc
        want[el < max(abs(m), abs(spin))] = 0
        assert np.abs(out[:, m + L - 1] - want).max() < 1e-11 * np.abs(want).max(), m


def test_real_signals(api, orc):
    for L in (16, 65, 140):
        flm = synth.random_flm(L, 0, seed=L, real=True)
        P = api.Plan(L, 0, reality=True)
        f = P.inverse(dev(flm)).cpu().numpy()
        f_ref = orc.s2_inverse(L, 0, orc.MW, flm)
        assert np.abs(f_ref.imag).max() < 1e-13
        assert rel(f, f_ref.real) < TOL
        back = P.forward(dev(f_ref.real.copy())).cpu().numpy()
        assert rel(back, flm) < TOL
        # input m<0 half is ignored
        junk = flm.copy(); junk[:, :L - 1] = 99.0
        # (not bit-equal: several l-tiles add into F_m(theta) with RED.ADD, whose order is not fixed)
        assert rel(P.inverse(dev(junk)).cpu().numpy(), f) < 1e-13


@pytest.mark.parametrize("L,N", [(4, 1), (8, 3), (16, 5), (33, 8), (40, 40)])
def test_so3_vs_oracle(api, orc, L, N):
    c = synth.random_flmn(L, N, seed=3 + L)
    P = api.Plan(L, N=N)
    f = P.inverse(dev(c)).cpu().numpy()
    f_ref = orc.so3_inverse(L, N, c)
    assert rel(f, f_ref) < TOL
    back = P.forward(dev(f_ref)).cpu().numpy()
    assert rel(back, c) < TOL
    assert rel(back, orc.so3_forward(L, N, f_ref)) < TOL


def test_host_buffer_calls_match_device_calls(api):
    L, spin = 50, 1
    flm = synth.random_flm(L, spin, seed=5)
    f_dev = api.s2_inverse(dev(flm), L, spin).cpu().numpy()
    f_host = api.s2_inverse_host(flm, L, spin)
    assert np.abs(f_host - f_dev).max() < 1e-13 * np.abs(f_dev).max()      # atomics order may differ in the last bits
    back = api.s2_forward_host(f_host, L, spin)
    assert rel(back, flm) < TOL
    c = synth.random_flmn(12, 3, seed=1)
    assert rel(api.so3_forward_host(api.so3_inverse_host(c, 12, 3), 12, 3), c) < TOL


@pytest.mark.parametrize("L,spin,sampling", [(1024, 2, "mw"), (1030, 0, "mw"), (1031, 1, "mwss"), (1025, 0, "mw")])
def test_host_buffer_calls_overlap_copies_in_ring_chunks(api, L, spin, sampling):
    """From L = 1024 the host-buffer calls run the ring FFT stage in 8 / 4 / 2 ring chunks on the transform's stream while a copy stream
    moves the next (forward) or the previous (inverse) chunk over PCIe; ring counts that no such chunk count divides (L = 1025) take
    the plain path.  Same numbers as the device-buffer calls, pinned and pageable host memory alike, and twice in a row (buffer reuse)."""
    samp = api.MW if sampling == "mw" else api.MWSS
    flm = synth.random_flm(L, spin, seed=L)
    f_dev = api.s2_inverse(dev(flm), L, spin, sampling=samp).cpu().numpy()
    for rep in range(2):
        f_host = api.s2_inverse_host(flm, L, spin, sampling=samp)
        assert np.abs(f_host - f_dev).max() < 1e-13 * np.abs(f_dev).max()
        back = api.s2_forward_host(f_host, L, spin, sampling=samp)
        assert rel(back, flm) < TOL
    pinned = torch.from_numpy(f_dev).pin_memory().numpy()
    assert rel(api.s2_forward_host(pinned, L, spin, sampling=samp), flm) < TOL


def test_inputs_are_not_modified_and_errors_are_loud(api):
    L = 20
    flm = synth.random_flm(L, 0, seed=1)
    d = dev(flm)
    keep = d.clone()
    f = api.s2_inverse(d, L, 0)
    keepf = f.clone()
    api.s2_forward(f, L, 0)
    torch.cuda.synchronize()
    assert torch.equal(d, keep) and torch.equal(f, keepf)
    with pytest.raises(ValueError):
        api.s2_inverse(d[:, :-1].contiguous(), L, 0)
    with pytest.raises(Exception):
        api.Plan(8, 9)


# HEALPix: ring FFTs of variable length with phase shift, periodic extension / folding of F_m.
# nside = 1 has no polar-cap rings; L > 4 nside - ... exercises aliasing (m >= nphi) on every ring; L = 2 nside is config 3's ratio.
@pytest.mark.parametrize("nside,L,spin,real", [(1, 3, 0, False), (2, 4, 0, True), (2, 9, 0, False), (4, 8, 0, True), (4, 11, 2, False),
                                               (8, 16, 0, True), (8, 16, -1, False), (16, 32, 0, True), (16, 40, 0, False), (32, 64, 0, True)])
def test_healpix_vs_oracle(api, orc, nside, L, spin, real):
    flm = synth.random_flm(L, spin, seed=nside + L, sigma=synth.SIGMA_RED, real=real)
    P = api.Plan(L, spin, sampling=api.HEALPIX, nside=nside, reality=real)
    f = P.inverse(dev(flm)).cpu().numpy()
    f_ref = orc.s2_inverse(L, spin, orc.HEALPIX, flm, nside=nside)
    assert f.shape == (12 * nside * nside,)
    if real:
        assert np.abs(f_ref.imag).max() < 1e-13 * np.abs(f_ref).max()
        f_ref = f_ref.real.copy()
    assert rel(f, f_ref) < TOL
    # HEALPix has no sampling theorem: forward parity is against the oracle's forward of the same map
    back = P.forward(dev(f_ref)).cpu().numpy()
    want = orc.s2_forward(L, spin, orc.HEALPIX, f_ref.astype(np.complex128), nside=nside)
    assert rel(back, want) < TOL
    el = np.arange(L)[:, None]
    m = np.arange(-(L - 1), L)[None, :]
    assert np.all(back[(np.abs(m) > el) | (el < abs(spin))] == 0)


def test_healpix_north_star_call_uses_nside_L_over_2(api, orc):
    L = 16
    flm = synth.random_flm(L, 0, seed=2, sigma=synth.SIGMA_RED, real=True)
    f = api.s2_inverse(dev(flm), L, 0, sampling=api.HEALPIX, reality=True)
    assert tuple(f.shape) == (12 * 8 * 8,)
    assert rel(f.cpu().numpy(), orc.s2_inverse(L, 0, orc.HEALPIX, flm, nside=8).real) < TOL
    back = api.s2_forward(f, L, 0, sampling=api.HEALPIX, reality=True).cpu().numpy()
    assert rel(back, orc.s2_forward(L, 0, orc.HEALPIX, f.cpu().numpy().astype(np.complex128), nside=8)) < TOL


@pytest.mark.parametrize("fold", ["0", "1"])
@pytest.mark.parametrize("sampling,L,nside,real", [("mw", 8, 0, False), ("mw", 33, 0, False), ("mw", 130, 0, False), ("mw", 200, 0, True),
                                                   ("hp", 9, 2, False), ("hp", 24, 8, True), ("hp", 64, 32, False)])
def test_spin0_forward_with_and_without_north_south_fold(api, orc, fold, sampling, L, nside, real):
    """The spin-0 forward runs the recursion on the northern rings only when the plan enables the fold (default at large L):
    d^l_{m0}(pi - theta) = (-1)^{l+m} d^l_{m0}(theta).  Both paths against the oracle, element by element."""
    fold = fold == "1"
    if sampling == "mw":
        f = synth.random_map((L, 2 * L - 1), seed=L, real=real)
        P = api.Plan(L, 0, reality=real, fold=fold)
        want = orc.s2_forward(L, 0, orc.MW, project_mw_pole(f, 0).astype(np.complex128))
    else:
        f = synth.random_map((12 * nside * nside,), seed=L, real=real)
        P = api.Plan(L, 0, sampling=api.HEALPIX, nside=nside, reality=real, fold=fold)
        want = orc.s2_forward(L, 0, orc.HEALPIX, f.astype(np.complex128), nside=nside)
    assert rel(P.forward(dev(f)).cpu().numpy(), want) < TOL
    if sampling == "hp":      # HEALPix rings are symmetric on the inverse side too: F_m(theta) = E + O, F_m(pi - theta) = E - O
        flm = synth.random_flm(L, 0, seed=3 * L, sigma=synth.SIGMA_RED, real=real)
        ref = orc.s2_inverse(L, 0, orc.HEALPIX, flm, nside=nside)
        got = P.inverse(dev(flm)).cpu().numpy()
        assert rel(got, ref.real if real else ref) < TOL


@pytest.mark.parametrize("sym", ["0", "1"])
@pytest.mark.parametrize("L,real", [(1, False), (2, False), (8, False), (33, False), (64, False), (130, False), (200, True), (257, False)])
def test_mw_spin0_inverse_with_and_without_symmetric_rings(api, orc, sym, L, real):
    """MW spin-0 inverse either directly on the MW rings (SHT_OPT_NO_INVSYM; default below L = 2048), or (SHT_OPT_INVSYM; default from L = 2048) on the L midpoint rings (2j+1)pi/(2L) with the
    north-south fold followed by an exact FFT resampling of F_m(theta) to the MW rings.  Both against the oracle, element by element,
    through the full transform and through the theta-stage entry point."""
    flm = synth.random_flm(L, 0, seed=5 * L, real=real)
    P = api.Plan(L, 0, reality=real, invsym=sym == "1")
    ref = orc.s2_inverse(L, 0, orc.MW, flm)
    got = P.inverse(dev(flm)).cpu().numpy()
    assert rel(got, ref.real if real else ref) < TOL
    F = P.theta_inverse(dev(flm)).cpu().numpy()
    assert rel(F, orc.s2_theta_inverse_columns(L, 0, orc.MW, flm, np.arange(-(L - 1), L))) < TOL


@pytest.mark.parametrize("sym", [False, True])
@pytest.mark.parametrize("L,spin", [(2, 1), (3, -2), (9, 1), (33, 2), (64, -1), (65, 3), (130, -2), (200, 1), (257, 2)])
def test_mw_spin_inverse_with_two_passes_or_one_fold_pass_on_symmetric_rings(api, orc, sym, L, spin):
    """spin != 0 MW inverse: two passes (second index n and -n) on the MW rings (SHT_OPT_NO_INVSYM; default below L = 2048), or ONE fold pass
    on the L midpoint rings -- order +m at a ring, order -m at its mirror ring, d^l_{-m,n}(pi - theta) = (-1)^{l-n} d^l_{m,n}(theta), PAPER.md:236 --
    followed by the exact FFT resampling to the MW rings (SHT_OPT_INVSYM; default from L = 2048).  Both against the oracle, element by element,
    through the full transform and through the theta-stage entry point."""
    flm = synth.random_flm(L, spin, seed=3 * L + spin)
    P = api.Plan(L, spin, invsym=sym)
    assert rel(P.inverse(dev(flm)).cpu().numpy(), orc.s2_inverse(L, spin, orc.MW, flm)) < TOL
    F = P.theta_inverse(dev(flm)).cpu().numpy()
    assert rel(F, orc.s2_theta_inverse_columns(L, spin, orc.MW, flm, np.arange(-(L - 1), L))) < TOL


@pytest.mark.parametrize("pair", [False, True])
@pytest.mark.parametrize("L,spin,fold,real", [(1, 0, None, False), (2, 0, None, False), (9, 1, None, False), (33, 0, True, False), (64, -2, None, False),
                                              (130, 0, True, True), (131, 3, None, False), (200, 0, False, False)])
def test_mw_theta_ffts_with_one_or_two_orders_per_column(api, orc, pair, L, spin, fold, real):
    """The extension of F_m to the theta circle is even or odd about the poles, alternating with m, so the theta-direction
    FFTs of the forward upsampling and of the symmetric-ring inverse carry the orders m, m+1 as ONE column and split them afterwards
    (default); SHT_OPT_NO_PAIR keeps one order per column.  Both against the oracle, on raw white noise (forward) and through the
    symmetric-ring inverse (spin 0)."""
    f = synth.random_map((L, 2 * L - 1), seed=11 + L, real=real)
    P = api.Plan(L, spin, reality=real, fold=fold, pair=pair, invsym=True)
    want = orc.s2_forward(L, spin, orc.MW, project_mw_pole(f, spin).astype(np.complex128))
    assert rel(P.forward(dev(f)).cpu().numpy(), want) < TOL
    flm = synth.random_flm(L, spin, seed=2 * L + 1, real=real)
    ref = orc.s2_inverse(L, spin, orc.MW, flm)
    assert rel(P.inverse(dev(flm)).cpu().numpy(), ref.real if real else ref) < TOL


@pytest.mark.parametrize("nside,L,spin,real", [(4, 8, 0, True), (8, 16, 0, True), (8, 20, 2, False), (16, 32, 0, False)])
def test_healpix_iterative_refinement_vs_oracle(api, orc, nside, L, spin, real):
    """PAPER.md:172 "iterations are usually performed": flm <- flm + F (f - F^-1 flm), against the oracle's composition of its own
    F and F^-1, element by element; plus, at a larger size, the property that the map residual shrinks with every iteration."""
    flm = synth.random_flm(L, spin, seed=nside + L, sigma=synth.SIGMA_RED, real=real)
    f_ref = orc.s2_inverse(L, spin, orc.HEALPIX, flm, nside=nside)
    f_in = f_ref.real.copy() if real else f_ref
    P = api.Plan(L, spin, sampling=api.HEALPIX, nside=nside, reality=real)
    for niter in (0, 1, 3):
        got = P.forward_iter(dev(f_in), niter).cpu().numpy()
        want = orc.s2_forward_iter(L, spin, orc.HEALPIX, f_ref, niter, nside=nside)
        assert rel(got, want) < TOL, niter
    with pytest.raises(Exception):
        api.Plan(L, spin).forward_iter(dev(synth.random_map((L, 2 * L - 1), seed=1)), 1)


def test_healpix_iterative_refinement_residual_shrinks_at_size(api):
    nside, L = 128, 256
    flm = dev(synth.random_flm(L, 0, seed=3, sigma=synth.SIGMA_RED, real=True))
    P = api.Plan(L, 0, sampling=api.HEALPIX, nside=nside, reality=True)
    f = P.inverse(flm)
    res, err = [], []
    for niter in range(4):
        c = P.forward_iter(f, niter)
        res.append(float((f - P.inverse(c)).abs().max()))
        err.append(float((c - flm).abs().max() / flm.abs().max()))
    assert all(b < a for a, b in zip(res, res[1:])) and err[3] < err[0] / 10, (res, err)

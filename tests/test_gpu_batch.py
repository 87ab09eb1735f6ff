"""GPU parity of the batched path (BASELINE.json configs[4] second half): a batch of S^2 maps sharing
one recursion, contraction on FP64 tensor-core MMAs (csrc/theta_mma.cu).  Every map of the batch is compared with the
CPU oracle element by element at small sizes (several 64 x 128 tiles plus ragged tails in L, rings and batch), and at
the full size of the config (16 maps, L = 2048) on sampled rings / harmonic orders plus the exact MW round trip."""
import numpy as np
import pytest

from paper_2311_14670_b200 import synth
from mwpole import project_mw_pole

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
TOL = 1e-11


def rel(a, b, scale=None):
    return float(np.abs(a - b).max() / (np.abs(b).max() if scale is None else scale))


@pytest.fixture(scope="module")
def api():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2311_14670_b200 import api as A
    return A


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# batch sizes: 16 complex columns per group -> spin 0 complex (2 columns per map): 8 maps fill one group, 3 leave
# padding, 9 straddle two groups; spin != 0 (1 column per map and pass, two passes); real (1 column per map)
@pytest.mark.parametrize("L,spin,batch,real", [(8, 0, 2, False), (33, 0, 3, False), (64, 0, 8, False), (130, 0, 9, False),
                                               (200, 0, 16, False), (48, 2, 5, False), (131, -2, 17, False), (65, 1, 16, False),
                                               (96, 0, 4, True), (257, 0, 2, False)])
def test_batched_s2_vs_oracle(api, orc, L, spin, batch, real):
    flm = np.stack([synth.random_flm(L, spin, seed=100 * L + b, real=real) for b in range(batch)])
    P = api.Plan(L, spin, reality=real, batch=batch)
    f = P.inverse(dev(flm)).cpu().numpy()
    f_ref = np.stack([orc.s2_inverse(L, spin, orc.MW, flm[b]) for b in range(batch)])
    if real:
        assert np.abs(f_ref.imag).max() < 1e-12 * np.abs(f_ref).max()
        f_ref = np.ascontiguousarray(f_ref.real)
    assert rel(f, f_ref) < TOL
    back = P.forward(dev(f_ref)).cpu().numpy()
    assert rel(back, flm) < TOL                                   # sampling theorem: exact round trip (pin 6)
    for b in (0, batch - 1):
        assert rel(back[b], orc.s2_forward(L, spin, orc.MW, f_ref[b].astype(np.complex128))) < TOL
    # coefficients outside the support are exact zeros
    el = np.arange(L)[:, None]
    m = np.arange(-(L - 1), L)[None, :]
    assert np.all(back[:, (np.abs(m) > el) | (el < abs(spin))] == 0)


def test_batched_equals_single_map_plans(api):
    """The batched kernels and the single-map kernels run the same recursion: results agree to rounding."""
    L, spin, batch = 192, 0, 6
    flm = np.stack([synth.random_flm(L, spin, seed=b) for b in range(batch)])
    Pb, P1 = api.Plan(L, spin, batch=batch), api.Plan(L, spin)
    fb = Pb.inverse(dev(flm))
    f1 = torch.stack([P1.inverse(dev(flm[b])) for b in range(batch)])
    assert float((fb - f1).abs().max() / f1.abs().max()) < 1e-13
    g = synth.random_map((batch, L, 2 * L - 1), seed=5)
    cb = Pb.forward(dev(g))
    c1 = torch.stack([P1.forward(dev(g[b])) for b in range(batch)])
    assert float((cb - c1).abs().max() / c1.abs().max()) < 1e-13


def test_config5b_batch16_L2048(api, orc):
    """configs[4], second half: 16 maps at L = 2048, spin 0, MW, sigma_l = 1/(l+1), seeds 4+b."""
    L, batch = 2048, 16
    flm = np.stack([synth.random_flm(L, 0, seed=4 + b, sigma=synth.SIGMA_RED) for b in range(batch)])
    P = api.Plan(L, 0, batch=batch)
    d = dev(flm)
    f = P.inverse(d)
    back = P.forward(f)
    assert float((back - d).abs().max() / d.abs().max()) < TOL       # exact round trip for every map
    rings = np.array([0, 3, 1000, 2046, 2047])
    for b in (0, 7, 15):
        rows = orc.s2_inverse_rings(L, 0, orc.MW, flm[b], rings)
        scale = max(np.abs(r).max() for r in rows)
        fb = f[b].cpu().numpy()
        for r, row in zip(rings, rows):
            assert rel(fb[r], row, scale) < TOL, (b, r)
    # forward of white-noise maps against the oracle on sampled orders m
    g = synth.random_map((batch, L, 2 * L - 1), seed=21)        # raw white noise to the GPU; the oracle gets the projected pole ring
    got = P.forward(dev(g))
    g = project_mw_pole(g, 0)
    ms = np.array([-(L - 1), -1000, -1, 0, 1, 2, 777, L - 1])
    for b in (0, 15):
        want = orc.s2_forward_columns(L, 0, orc.MW, g[b], ms)
        sc = np.abs(want).max()
        gb = got[b].cpu().numpy()
        for m, col in zip(ms, want):
            assert rel(gb[:, m + L - 1], col, sc) < TOL, (b, m)


@pytest.mark.parametrize("fold", ["0", "1"])
@pytest.mark.parametrize("L,batch,real", [(8, 2, False), (33, 3, False), (130, 9, False), (200, 16, False), (96, 4, True)])
def test_batched_spin0_forward_with_and_without_fold(api, orc, fold, L, batch, real):
    """Batched spin-0 forward with the north-south fold forced on / off (default: on at large L): recursion on the northern rings,
    even / odd l+m rows contract with the E / O column sets (theta_mma.cu FOLD).  White-noise maps, every map against the oracle."""
    g = synth.random_map((batch, L, 2 * L - 1), seed=7 * L, real=real)
    P = api.Plan(L, 0, reality=real, batch=batch, fold=fold == "1")
    got = P.forward(dev(g)).cpu().numpy()
    g = project_mw_pole(g, 0)
    for b in range(batch):
        assert rel(got[b], orc.s2_forward(L, 0, orc.MW, g[b].astype(np.complex128))) < TOL, b


@pytest.mark.parametrize("kind", ["hp", "mwss", "dh", "gl", "f32", "f32s2"])
def test_batches_without_batched_kernels_run_map_by_map(api, orc, kind):
    """A batch on a sampling (or dtype) the shared-recursion DMMA kernels do not serve is accepted and transformed map by map through the
    single-map kernels: same array layout (leading [batch] axis), every map against the oracle."""
    L, B = 40, 3
    if kind in ("f32", "f32s2"):               # (f32s2: fp32 arrays around the fp64 kernels, spin 2)
        spin = 2 if kind == "f32s2" else 0
        P = api.Plan(L, spin, batch=B, dtype="f32")
        os_, okw, tol = orc.MW, {}, 1e-4
    else:
        gs, os_ = {"hp": (api.HEALPIX, orc.HEALPIX), "mwss": (api.MWSS, orc.MWSS), "dh": (api.DH, orc.DH), "gl": (api.GL, orc.GL)}[kind]
        nside = 8 if kind == "hp" else 0
        spin, tol = 2, 1e-12
        P = api.Plan(L, spin, sampling=gs, nside=nside, batch=B)
        okw = dict(nside=nside) if kind == "hp" else {}
    flm = np.stack([synth.random_flm(L, spin, seed=50 + b) for b in range(B)])
    x = flm.astype(np.complex64) if kind in ("f32", "f32s2") else flm
    f = P.inverse(dev(x))
    assert tuple(f.shape)[0] == B
    for b in range(B):
        ref = orc.s2_inverse(L, spin, os_, flm[b], **okw)
        assert float(np.abs(f[b].cpu().numpy() - ref).max() / np.abs(ref).max()) < tol
    back = P.forward(f).cpu().numpy()
    for b in range(B):
        want = orc.s2_forward(L, spin, os_, f[b].cpu().numpy().astype(np.complex128), **okw)
        assert float(np.abs(back[b] - want).max() / np.abs(want).max()) < tol

"""s2_theta_inverse_noalloc (include/b200sht.h): the allocation-free entry point against the existing plan path
(Plan.theta_inverse, the fused on-the-fly kernels) on the same seeded coefficients, same tolerance as test_gpu_parity.py.

Collected last on purpose (file name): the suite runs with pytest -x, so a failure here hides nothing.  Calls are made back to
back on one stream and at different sizes, so that each call finds the static table full of the previous call's d-functions."""
import ctypes as C

import numpy as np
import pytest

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


def rings(sampling, L):
    """Colatitudes of the inverse rings of the plan path (Sec. 2.5: MW Eq. 34, MWSS, DH Eq. 35)."""
    if sampling == "mw":
        return np.array([(2 * t + 1) * np.pi / (2 * L - 1) for t in range(L)])          # last ring at theta = pi
    if sampling == "mwss":
        return np.array([t * np.pi / L for t in range(L + 1)])                             # both poles
    return np.array([(2 * t + 1) * np.pi / (4 * L) for t in range(2 * L)])                # dh


def plan_path(api, L, spin, sampling, flm):
    code = {"mw": api.MW, "mwss": api.MWSS, "dh": api.DH}[sampling]
    P = api.Plan(L, spin, sampling=code)
    assert P.ntheta(False) == len(rings(sampling, L))
    return P.theta_inverse(flm).cpu().numpy()


CASES = [(64, 0, "dh"),      # 127 * 128 * 64 table entries: 99 % of the static scratch
         (33, -1, "mwss"),   # smaller table inside the previous call's, both pole rings (Eq. 28 / 29)
         (48, 2, "mw"),      # two recursion passes per ring (spin != 0), pole ring at theta = pi
         (64, 0, "dh")]      # the first case again, after two other tables


def test_noalloc_matches_plan_path_on_consecutive_calls(api):
    got, want = [], []
    for i, (L, spin, sampling) in enumerate(CASES):
        flm = torch.from_numpy(synth.random_flm(L, spin, seed=11 + i)).cuda()
        want.append(plan_path(api, L, spin, sampling, flm))
        th = rings(sampling, L)
        out = torch.full((2 * L - 1, len(th)), float("nan"), dtype=torch.complex128, device="cuda")
        # two calls in a row into the same output, nothing in between
        api.theta_inverse_noalloc(flm, L, spin, th, out=out)
        first = out.clone()
        api.theta_inverse_noalloc(flm, L, spin, th, out=out)
        torch.cuda.synchronize()
        assert torch.equal(first, out), "second call differs from the first"
        got.append(out.cpu().numpy())
    for (L, spin, sampling), g, w in zip(CASES, got, want):
        assert np.all(np.isfinite(g.view(np.float64))), (L, spin, sampling)
        assert rel(g, w) < TOL, (L, spin, sampling, rel(g, w))


def test_noalloc_matches_oracle_columns(api, orc):
    L, spin = 40, -2
    flm = synth.random_flm(L, spin, seed=5)
    ms = [-(L - 1), -7, -2, 0, 1, 2, 3, L - 1]
    ref = orc.s2_theta_inverse_columns(L, spin, orc.MW, flm, ms)
    out = api.theta_inverse_noalloc(torch.from_numpy(flm).cuda(), L, spin, rings("mw", L)).cpu().numpy()
    assert rel(out[[m + L - 1 for m in ms]], ref) < TOL


def test_noalloc_uses_no_device_memory(api):
    L, spin = 32, 1
    th = rings("mw", L)
    flm = torch.from_numpy(synth.random_flm(L, spin, seed=3)).cuda()
    out = torch.empty((2 * L - 1, L), dtype=torch.complex128, device="cuda")
    api.theta_inverse_noalloc(flm, L, spin, th, out=out)          # first call: module load, symbol lookup
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        api.theta_inverse_noalloc(flm, L, spin, th, out=out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, f"device memory shrank by {free0 - free1} bytes across allocation-free calls"


def test_noalloc_rejects_sizes_beyond_the_static_scratch(api):
    from paper_2311_14670_b200 import _lib
    lib = _lib.lib()
    flm = torch.zeros((128, 255), dtype=torch.complex128, device="cuda")
    out = torch.zeros((255, 128), dtype=torch.complex128, device="cuda")
    err = C.create_string_buffer(512)

    def call(L, spin, th):
        th = np.ascontiguousarray(th, dtype=np.float64)
        return lib.s2_theta_inverse_noalloc(L, spin, len(th), th.ctypes.data_as(C.POINTER(C.c_double)), C.c_void_p(flm.data_ptr()),
                                            C.c_void_p(out.data_ptr()), None, err, len(err))

    assert call(128, 0, rings("mw", 128)) == 2 and b"exceed the fixed scratch" in err.value          # SHT_EUNSUPPORTED
    assert call(65, 0, rings("dh", 65)) == 2 and b"SHT_NOALLOC_MAX_RINGS" in err.value               # 130 rings
    assert call(8, 8, rings("mw", 8)) == 1 and b"spin" in err.value                                   # SHT_EINVAL
    assert call(8, 0, np.array([0.1, 4.0])) == 1 and b"[0, pi]" in err.value
    assert (2 * 64 - 1) * 128 * 64 * 8 <= _lib.SHT_NOALLOC_SCRATCH_BYTES < (2 * 65 - 1) * 128 * 65 * 8
    torch.cuda.synchronize()
    assert torch.count_nonzero(out) == 0                                                              # nothing was launched
    with pytest.raises(_lib.ShtError, match="exceed the fixed scratch"):
        api.theta_inverse_noalloc(flm, 128, 0, rings("mw", 128))

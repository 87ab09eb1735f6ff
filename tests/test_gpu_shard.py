"""Ring-sharded transforms on ONE GPU: a plan told to serve share k of K of the kernel
rings returns a partial flm (forward) or a map with only its rings filled (inverse); the sum over the K shards must be the
unsharded transform, and the shares must be the balanced partition the multi-GPU driver (bench.py --shard rings,
paper_2311_14670_b200/ranks.py) assumes.  No collective is exercised here: the sum over shards stands in for the all-reduce."""
import numpy as np
import pytest

from paper_2311_14670_b200 import synth
from paper_2311_14670_b200.ranks import split_range

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
TOL = 1e-12


@pytest.fixture(scope="module")
def api():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2311_14670_b200 import api as A
    return A


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def relt(a, b):
    return float((a - b).abs().max() / b.abs().max())


@pytest.mark.parametrize("K", [2, 3, 8])
@pytest.mark.parametrize("kind,L,spin,kw", [("mw", 130, 0, {}), ("mw", 200, 2, {}), ("mw", 257, 0, dict(fold=True)), ("mw", 96, 0, dict(reality=True)),
                                            ("mwss", 130, 1, {}), ("dh", 64, 0, {}), ("gl", 131, -2, {}), ("hp", 64, 0, dict(nside=32, reality=True)),
                                            ("hp", 40, 2, dict(nside=16)),
                                            ("mw", 1100, 0, {}), ("dh", 1030, 1, {})])      # (L >= 1024: blocks start from the stored silent-head state)
def test_sum_over_ring_shards_is_the_transform(api, kind, L, spin, kw, K):
    samp = {"mw": api.MW, "mwss": api.MWSS, "dh": api.DH, "gl": api.GL, "hp": api.HEALPIX}[kind]
    real = kw.get("reality", False)
    P = api.Plan(L, spin, sampling=samp, invsym=False, **kw)
    flm = dev(synth.random_flm(L, spin, seed=L, real=real))
    g = dev(synth.random_map(P.map_shape, seed=L + 1, real=real))
    full_f, full_c = P.inverse(flm).clone(), P.forward(g).clone()
    acc_f, acc_c = torch.zeros_like(full_f), torch.zeros_like(full_c)
    for fwd in (False, True):
        nth = P.shard_range(fwd)[1]
        spans = []
        for k in range(K):
            P.set_shard(k, K)
            spans.append(P.shard_range(fwd))
            assert spans[-1] == split_range(nth, K, k)            # the partition the host-side rank logic assumes
        P.set_shard(0, 1)
        assert spans[0][0] == 0 and spans[-1][1] == nth and all(spans[i][1] == spans[i + 1][0] for i in range(K - 1))
    filled = torch.zeros(full_f.shape, dtype=torch.int32, device=full_f.device)
    for k in range(K):
        P.set_shard(k, K)
        part = P.inverse(flm)
        filled += (part != 0).to(torch.int32)
        acc_f += part
        acc_c += P.forward(g)
    P.set_shard(0, 1)
    assert relt(acc_f, full_f) < TOL and relt(acc_c, full_c) < TOL
    assert int(filled.max()) <= 1                                  # every sample of the map is produced by exactly one shard
    assert relt(P.inverse(flm), full_f) < 1e-14                    # (0, 1) restores the whole transform


def test_so3_shards_and_unsupported_plans(api):
    L, N, K = 24, 3, 2
    c = dev(synth.random_flmn(L, N, seed=1))
    P = api.Plan(L, N=N)
    full = P.inverse(c).clone()
    back = P.forward(full).clone()
    acc, accb = torch.zeros_like(full), torch.zeros_like(back)
    for k in range(K):
        P.set_shard(k, K)
        acc += P.inverse(c)
        accb += P.forward(full)
    assert relt(acc, full) < TOL and relt(accb, back) < TOL
    from paper_2311_14670_b200._lib import ShtError
    for kw in (dict(batch=2), dict(dtype="f32"), dict(adjoint=True), dict(invsym=True)):
        with pytest.raises(ShtError):
            api.Plan(32, 0, **kw).set_shard(0, 2)
    with pytest.raises(ShtError):
        P.set_shard(2, 2)

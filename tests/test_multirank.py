"""World-size-2 `gloo` tests (CPU) of the host-side rank logic used by `bench.py --gpus N`.

The path shards over independent problems: no data-path collective; what the ranks exchange is the barrier and the
MAX of their elapsed times.  The ring-sharded variant additionally needs a balanced ring split and one
SUM all-reduce of partial f_lm: both are exercised here with the CPU oracle standing in for the per-rank transform
(the partial forward of a ring subset is the oracle's quadrature sum restricted to those rings).
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    if root not in sys.path:
        sys.path.insert(0, root)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2311_14670_b200 import ranks, synth
    import oracle
    R = ranks.Ranks(backend="gloo")
    out = {"rank": R.rank, "world": R.world}
    # (1) distinct seeded problems per rank
    flm = synth.random_flm(12, 0, seed=R.seed(5))
    out["flm_sum"] = complex(flm.sum())
    # (2) timing reduction: max over ranks, aggregate throughput
    R.barrier()
    t = R.max_over_ranks(10.0 + 5.0 * rank)
    out["tmax"] = t
    out["value"] = R.throughput(1, 4, t)
    # (3) ring-sharded inverse: each rank synthesises its rings only; the union is the full map (no collective)
    L, spin = 12, 1
    c = synth.random_flm(L, spin, seed=3)
    a, b = R.ring_range(L)
    rows = oracle.s2_inverse_rings(L, spin, oracle.MW, c, np.arange(a, b))
    part = torch.zeros((L, 2 * L - 1), dtype=torch.complex128)
    for i, r in enumerate(range(a, b)):
        part[r] = torch.from_numpy(rows[i])
    buf = torch.view_as_real(part).contiguous()
    R.sum_over_ranks(buf)                       # disjoint rows: the sum assembles the map
    out["map"] = torch.view_as_complex(buf).numpy()
    out["range"] = (a, b)
    # (4) the code path of `bench.py --gpus N --shard rings`: sharded.ShardedTransform over this process group, with a CPU stand-in
    # for the ring-sharded plan (the oracle restricted to the rank's rings; the library's share rule is ranks.split_range)
    from paper_2311_14670_b200.sharded import ShardedTransform
    ST = ShardedTransform(OraclePlan(oracle, L, spin), R)
    cc = torch.from_numpy(c)
    f_full = ST.inverse(cc, gather=True)
    out["sharded_map"] = f_full.numpy().copy()
    out["sharded_back"] = ST.forward(f_full).numpy().copy()
    R.finish()
    q.put(out)


class OraclePlan:
    """CPU stand-in for a ring-sharded api.Plan (MW): serves the ranks.split_range share of the rings with the oracle.  inverse:
    the rank's rings of the map, zeros elsewhere; forward: Eq. 30 restricted to the rank's share of the 2L quadrature rings."""

    def __init__(self, oracle, L, spin):
        self.o, self.L, self.spin, self.rank, self.n = oracle, L, spin, 0, 1

    def set_shard(self, rank, n):
        self.rank, self.n = rank, n

    def inverse(self, flm, out=None):
        from paper_2311_14670_b200.ranks import split_range
        L = self.L
        a, b = split_range(L, self.n, self.rank)
        f = torch.zeros((L, 2 * L - 1), dtype=torch.complex128)
        rows = self.o.s2_inverse_rings(L, self.spin, self.o.MW, flm.numpy(), np.arange(a, b))
        for i, r in enumerate(range(a, b)):
            f[r] = torch.from_numpy(rows[i])
        return f

    def forward(self, f, out=None):
        from paper_2311_14670_b200.ranks import split_range
        o, L, s = self.o, self.L, self.spin
        ms = np.arange(-(L - 1), L)
        # full staging on every rank (ring DFT, extension, upsampling to the oracle's 2L quadrature rings), theta step on the share
        U = np.zeros((2 * L - 1, 2 * L), complex)
        Fm = np.fft.fft(f.numpy(), axis=1)
        T, sg = 2 * L - 1, (-1.0) ** (ms + s)
        t = np.arange(T)
        u = np.arange(2 * L)
        for i, m in enumerate(ms):
            col = Fm[:, m % T]
            ext = np.concatenate([col, sg[i] * col[L - 2::-1]])
            mp = np.arange(-(L - 1), L)
            Fmm = (ext[None, :] * np.exp(-1j * np.pi * mp[:, None] * (2 * t[None, :] + 1) / T)).sum(1) / T
            U[i] = (Fmm[None, :] * np.exp(1j * np.pi * mp[None, :] * (2 * u[:, None] + 1) / (4 * L - 1))).sum(1)
        tab = o.ring_table(o.MW_QUAD, L)
        W = U * np.asarray(tab["weight"], float)[None, :]
        a, b = split_range(2 * L, self.n, self.rank)
        W[:, :a] = 0
        W[:, b:] = 0
        return torch.from_numpy(np.ascontiguousarray(o.s2_theta_forward_columns(L, s, o.MW_QUAD, W, ms).T))


@pytest.mark.timeout(300)
def test_two_ranks_gloo():
    from paper_2311_14670_b200 import synth
    import oracle
    oracle.lib()                                 # build once before forking workers
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=240) for _ in procs), key=lambda d: d["rank"])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [d["world"] for d in res] == [2, 2]
    # distinct problems per rank, reproducible from the seed rule
    assert res[0]["flm_sum"] != res[1]["flm_sum"]
    assert res[1]["flm_sum"] == complex(synth.random_flm(12, 0, seed=6).sum())
    # max over ranks and whole-job throughput
    assert res[0]["tmax"] == res[1]["tmax"] == 15.0
    assert res[0]["value"] == pytest.approx(2 * 4 / 15e-3)
    # ring split is a partition, and the assembled map equals the single-process oracle map
    assert res[0]["range"] == (0, 6) and res[1]["range"] == (6, 12)
    full = oracle.s2_inverse(12, 1, oracle.MW, synth.random_flm(12, 1, seed=3))
    for d in res:
        assert np.abs(d["map"] - full).max() <= 1e-14 * np.abs(full).max()
    # the sharded transform pair (bench.py --shard rings): assembled map and summed partial flm on EVERY rank
    c = synth.random_flm(12, 1, seed=3)
    for d in res:
        assert np.abs(d["sharded_map"] - full).max() <= 1e-14 * np.abs(full).max()
        assert np.abs(d["sharded_back"] - c).max() <= 1e-13 * np.abs(c).max()          # sampling theorem: the round trip is exact


def test_split_range_is_a_balanced_partition():
    from paper_2311_14670_b200.ranks import split_range
    for n in (0, 1, 7, 8, 1023, 4095):
        for parts in (1, 2, 3, 8):
            spans = [split_range(n, parts, i) for i in range(parts)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(spans[i][1] == spans[i + 1][0] for i in range(parts - 1))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1


def test_single_process_defaults():
    from paper_2311_14670_b200 import ranks
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    R = ranks.Ranks(backend="gloo")
    assert (R.rank, R.world, R.dist) == (0, 1, None)
    assert R.max_over_ranks(3.5) == 3.5 and R.seed(4) == 4
    assert R.throughput(1, 10, 100.0) == pytest.approx(100.0)

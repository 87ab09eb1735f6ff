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
    R.finish()
    q.put(out)


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

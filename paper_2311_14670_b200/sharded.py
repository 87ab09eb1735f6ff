"""One transform spread over the ranks of a process group (ring shards; include/b200sht.h sht_plan_set_shard).

Host-side plumbing only: which rank serves which rings is decided inside the library (balanced contiguous shares, the rule of
ranks.split_range); this module adds the two collectives the method needs on top of a ring-sharded plan:

    inverse : flm replicated on every rank -> each rank fills its rings of the map.  No collective is needed to OWN the rings;
              `gather=True` additionally assembles the full map on every rank (SUM all-reduce of disjoint rings), which the MW /
              MWSS forward transform needs as input because its theta-upsampling mixes rings.
    forward : each rank integrates over its quadrature rings -> partial flm -> ONE SUM all-reduce of L (2L-1) complex numbers.

`plan` is anything with set_shard(rank, n), inverse(flm, out=) and forward(f, out=) on torch tensors -- api.Plan on a GPU (NCCL), or
a CPU stand-in in the gloo tests, so that the code that runs under `bench.py --gpus N --shard rings` is the code that is tested.
"""
import torch


def _as_real(t):
    return torch.view_as_real(t) if t.is_complex() else t


class ShardedTransform:
    def __init__(self, plan, ranks):
        self.plan, self.ranks = plan, ranks
        plan.set_shard(ranks.rank, ranks.world)

    def inverse(self, flm, out=None, gather=True):
        f = self.plan.inverse(flm, out=out)
        if gather:
            self.ranks.sum_over_ranks(_as_real(f))      # rings are disjoint across ranks: the sum assembles the map
        return f

    def forward(self, f, out=None):
        c = self.plan.forward(f, out=out)
        self.ranks.sum_over_ranks(_as_real(c))          # partial quadrature sums -> the transform
        return c

    def allreduce_bytes(self, flm, f, gather=True):
        """bytes each rank contributes to the collectives of one inverse + forward pair"""
        return flm.numel() * flm.element_size() + (f.numel() * f.element_size() if gather else 0)

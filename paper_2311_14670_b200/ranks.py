"""Host-side rank plumbing for multi-GPU runs (one process per GPU, torch.distributed).

The transforms shard over *independent problems* (DESIGN.md "Multi-GPU"): every rank transforms its own seeded field,
there is no data-path collective; the only communication is the barrier and the max-over-ranks of the elapsed device
time.  This module holds that logic so that it can be exercised with the `gloo` backend on CPU
(tests/test_multirank.py); it contains none of the method's arithmetic.
"""
import os

import torch


class Ranks:
    """Rank / world bookkeeping read from the torchrun environment (RANK, LOCAL_RANK, WORLD_SIZE, MASTER_*)."""

    def __init__(self, backend="nccl", init=True):
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.backend = backend
        self.dist = None
        if self.world > 1 and init:
            import torch.distributed as dist
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            kw = {}
            if backend == "nccl":
                kw["device_id"] = torch.device(f"cuda:{self.local_rank}")
            if not dist.is_initialized():
                dist.init_process_group(backend, rank=self.rank, world_size=self.world, **kw)
            self.dist = dist

    # -- work assignment --------------------------------------------------------------------------------------
    def seed(self, base_seed):
        """Weak scaling: rank r transforms the field drawn from seed base_seed + r (distinct problems)."""
        return int(base_seed) + self.rank

    def ring_range(self, nrings):
        """Contiguous, balanced share of `nrings` iso-latitude rings for this rank (ring-sharded variant, SURVEY
        8(e): every ring costs the same number of d-steps).  Returns (first, last+1)."""
        return split_range(nrings, self.world, self.rank)

    # -- collectives on scalars (timing only) -----------------------------------------------------------------
    def barrier(self, device_sync=None):
        if self.dist is not None:
            self.dist.barrier()
        if device_sync is not None:
            device_sync()

    def max_over_ranks(self, value, device=None):
        """MAX over ranks of a host float (the elapsed device time of the timed region)."""
        if self.dist is None:
            return float(value)
        t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(self, tensor):
        """In-place SUM all-reduce of a tensor (ring-sharded forward: partial f_lm of each rank's rings)."""
        if self.dist is not None:
            self.dist.all_reduce(tensor, op=self.dist.ReduceOp.SUM)
        return tensor

    def throughput(self, units_per_rank_per_step, steps, total_ms_max):
        """Whole-job units per second: all ranks' units divided by the slowest rank's time."""
        return self.world * units_per_rank_per_step * steps / (total_ms_max * 1e-3)

    def finish(self):
        if self.dist is not None:
            self.dist.barrier()
            self.dist.destroy_process_group()
            self.dist = None


def split_range(n, parts, i):
    """[first, last) of part i when n items are split into `parts` contiguous shares differing by at most one."""
    if not (0 <= i < parts):
        raise ValueError("part index out of range")
    q, r = divmod(int(n), int(parts))
    first = i * q + min(i, r)
    return first, first + q + (1 if i < r else 0)

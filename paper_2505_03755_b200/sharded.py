"""Aux-sharded DF-JK across ranks: one process per GPU.

J and K are sums over the aux index P of terms that need only row P of B (rho_P is local to P), so
rank r keeps the contiguous aux rows [lo_r, hi_r) resident (the paper's "hashing" of blocks to GPUs,
PAPER.md:257), runs the unchanged single-GPU path on its slice, and ONE sum all-reduce of the
nset x nao x nao partial J and K finishes the call -- on the devices, over NCCL/NVLink, instead of
the paper's serial accumulation on the CPU.  BASELINE.json's north_star is a
single-GPU build, so bench.py defaults to independent replicas; `bench.py --shard-aux` uses this
class.  Only marshalling and the collective live here; the arithmetic stays in the CUDA kernels.
"""
from __future__ import annotations

from typing import Callable, Optional, Tuple


def aux_range(naux: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous, balanced aux rows of `rank`: sizes differ by at most one, earlier ranks larger."""
    if world < 1 or not (0 <= rank < world) or naux < 0:
        raise ValueError("bad rank/world/naux")
    base, extra = divmod(naux, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


class AuxShardedJK:
    """get_jk over ranks that each hold a slice of the aux rows.

    local_get_jk(*args, **kw) -> (J, K): the partial results of this rank's slice as torch tensors
    (a `DFJK.get_jk` bound to a handle created on B[lo:hi]); either may be None.
    """

    def __init__(self, local_get_jk: Callable, group=None):
        import torch.distributed as dist
        self._local = local_get_jk
        self._dist = dist if dist.is_available() and dist.is_initialized() else None
        self._group = group

    def get_jk(self, *args, **kw):
        J, K = self._local(*args, **kw)
        if self._dist is not None and self._dist.get_world_size(self._group) > 1:
            # stream-ordered after the local kernels (NCCL on the current stream); sums in rank order
            for t in (J, K):
                if t is not None:
                    self._dist.all_reduce(t, op=self._dist.ReduceOp.SUM, group=self._group)
        return J, K


def make_sharded(B_rows, nao: int, naux_total: int, rank: Optional[int] = None, world: Optional[int] = None, **opts):
    """Convenience for the GPU path: `B_rows` is this rank's slice B[lo:hi] (CUDA tensor);
    returns (AuxShardedJK, DFJK handle)."""
    import torch.distributed as dist
    from .api import DFJK
    rank = dist.get_rank() if rank is None else rank
    world = dist.get_world_size() if world is None else world
    lo, hi = aux_range(naux_total, rank, world)
    if int(B_rows.shape[0]) != hi - lo:
        raise ValueError(f"rank {rank} must hold aux rows [{lo}, {hi})")
    h = DFJK(B_rows, nao, **opts)
    return AuxShardedJK(h.get_jk), h

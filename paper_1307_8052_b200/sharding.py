"""Multi-GPU sharding of the chi0 accumulation (host logic only, no arithmetic of the method).

Transitions are independent ("no MPI communication required during the calculation"), so the work of
one q-point is split into units (k-point, block of occupied bands); every rank accumulates its units into private
accumulators S and the only exchange is one sum of S over ranks at the end of the q-point (NCCL all-reduce over
NVLink on GPUs; gloo in the CPU tests).  After the sum every rank holds the full S, so rpa_chi0_get / rpa_ec_q can
run anywhere (rpa_ec_q's frequencies could also be split, E_c(q) being a plain sum over frequencies).
"""
from __future__ import annotations

from typing import List, Tuple

Unit = Tuple[int, int, int]  # (k index, first occupied band, one-past-last occupied band)


def shard_units(n_k: int, n_occ: int, rank: int, world: int) -> List[Unit]:
    """Units of rank `rank`: whole k-points round-robin when there are at least `world` of them, otherwise each
    k-point's occupied bands are cut into ceil(world / n_k) nearly equal blocks first.  Every (k, band) belongs to
    exactly one rank; ranks may get no unit when there is less work than ranks."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank / world")
    if n_k < 1 or n_occ < 1:
        return []
    split = 1 if n_k >= world else min(n_occ, -(-world // n_k))
    units: List[Unit] = []
    for k in range(n_k):
        base, rem = divmod(n_occ, split)
        lo = 0
        for b in range(split):
            hi = lo + base + (1 if b < rem else 0)
            units.append((k, lo, hi))
            lo = hi
    return [u for i, u in enumerate(units) if i % world == rank]


def allreduce_accumulators(S, group=None):
    """In-place sum over ranks of the accumulators (a complex128 tensor, CUDA for NCCL or CPU for gloo)."""
    import torch
    import torch.distributed as dist
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return S
    dist.all_reduce(torch.view_as_real(S), op=dist.ReduceOp.SUM, group=group)
    return S

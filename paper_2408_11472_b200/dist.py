"""Multi-GPU plumbing: the spectrum is a sum over scatterers, so
each rank accumulates a contiguous block of along-track rows into a partial T_u and ONE all-reduce of the
[G][N] complex64 grid per update joins them (the paper's host gather thread).  No arithmetic of
the method lives here: only the partition and the collective call (NCCL on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

import torch


def shard_rows(n_along: int, rank: int, world: int) -> tuple[int, int]:
    """Along-track rows [lo, hi) of rank `rank`: contiguous, disjoint, covering, sizes differ by at most 1."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    return n_along * rank // world, n_along * (rank + 1) // world


def shard_scatterers(scat: dict, n_cross: int, rank: int, world: int) -> dict:
    """This rank's slice of every SoA array (flat index = row * n_cross + column).  Row boundaries are
    multiples of n_cross, so 16-byte alignment is kept whenever n_cross is a multiple of 4."""
    if world == 1:
        return scat
    n = next(iter(scat.values())).numel()
    if n % n_cross:
        raise ValueError("scatterer count is not a multiple of n_cross")
    lo, hi = shard_rows(n // n_cross, rank, world)
    return {k: v[lo * n_cross:hi * n_cross].contiguous() for k, v in scat.items()}


def allreduce_spectrum(T: torch.Tensor, group=None) -> torch.Tensor:
    """Sums the partial spectra of all ranks in place (the one exchange step of an update).  T: complex64
    [G][N], or its float32 view [G][N][2] (Sim.spectrum_view: a view of the library's workspace)."""
    import torch.distributed as dist
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return T
    dist.all_reduce(torch.view_as_real(T) if T.is_complex() else T, op=dist.ReduceOp.SUM, group=group)
    return T

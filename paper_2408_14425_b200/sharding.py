"""Wavelength sharding across ranks.

Every wavelength is an independent formal solution, so the path shards by
contiguous wavelength blocks with no exchange during the solve.  Only host-side logic lives here:
the block partition, the optional all-gather of per-wavelength J and the all-reduce of Jbar, both
through torch.distributed (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations


def wavelength_block(nlambda: int, rank: int, world: int) -> tuple[int, int]:
    """[l0, l1) of rank `rank`: contiguous, sizes differ by at most one, empty if nlambda < world."""
    assert 0 <= rank < world and nlambda >= 0
    base, rem = divmod(nlambda, world)
    l0 = rank * base + min(rank, rem)
    return l0, l0 + base + (1 if rank < rem else 0)


def shard_atmosphere(atm, rank: int, world: int):
    """The rank's slice of an `atmospheres.Atmosphere` (copies: the C ABI wants contiguous planes)."""
    import copy
    import numpy as np
    l0, l1 = wavelength_block(atm.nlambda, rank, world)
    out = copy.copy(atm)
    out.nlambda = l1 - l0
    if getattr(atm, "line", None) is not None:
        # moving line: the six per-cell parameters are the same on every rank, the rank's block is its wavelengths x_l
        out.xl = np.ascontiguousarray(atm.xl[l0:l1])
    else:
        out.chi = np.ascontiguousarray(atm.chi[:, :, l0:l1])
        out.eta = np.ascontiguousarray(atm.eta[:, :, l0:l1])
    out.I_below = atm.I_below[l0:l1].copy()
    out.I_above = atm.I_above[l0:l1].copy()
    out.weights = atm.weights[l0:l1].copy()
    return out


def allreduce_jbar(jbar_local):
    """Jbar = sum over ranks of the ranks' weighted partial sums: one all-reduce of nx*ny floats."""
    import torch.distributed as dist
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(jbar_local, op=dist.ReduceOp.SUM)
    return jbar_local


def allgather_j(j_local, nlambda: int):
    """Per-wavelength J [ny][nx][L] on every rank from the ranks' blocks (blocks may differ by one)."""
    import torch
    import torch.distributed as dist
    if not dist.is_initialized() or dist.get_world_size() == 1:
        return j_local
    world = dist.get_world_size()
    ny, nx = j_local.shape[:2]
    width = max(wavelength_block(nlambda, r, world)[1] - wavelength_block(nlambda, r, world)[0] for r in range(world))
    pad = torch.zeros(ny, nx, width, dtype=j_local.dtype, device=j_local.device)
    pad[:, :, : j_local.shape[2]] = j_local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    cols = []
    for r, p in enumerate(parts):
        l0, l1 = wavelength_block(nlambda, r, world)
        cols.append(p[:, :, : l1 - l0])
    return torch.cat(cols, dim=2)

"""One process per GPU: k-points (or cells) of one band-structure job split over the ranks of a torch.distributed group.

SURVEY 8(e) / PAPER.md:205 (every k-point is an independent eigenproblem once Phi^-1 and the factor of Psi exist; the
paper notes the same for CPU cores).  The path has no exchange step, so there is no data-path collective: every rank
assembles its own copy of the cell (``bs_assemble`` is a few ms) or only its own cells, solves a CONTIGUOUS range of
k-points (configs 1-3, 5) or of cells (config 4), and one all-gather of ``nk x nbands`` doubles puts the whole result on
every rank.  This module only does index arithmetic, argument marshalling and that collective; every arithmetic step of
the path runs in the kernels behind ``bs_assemble_batch`` / ``bs_bands_batch``.
"""
from __future__ import annotations

from typing import List, Sequence, Tuple

import numpy as np


def shard_range(n: int, world: int, rank: int) -> Tuple[int, int]:
    """Contiguous range [lo, hi) of rank ``rank`` when n units are split over ``world`` ranks: the first n % world
    ranks get one unit more.  Ranges are disjoint, ordered by rank, and cover [0, n)."""
    if world < 1 or not (0 <= rank < world) or n < 0:
        raise ValueError("shard_range: bad arguments")
    base, extra = divmod(n, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_counts(n: int, world: int) -> List[int]:
    return [shard_range(n, world, r)[1] - shard_range(n, world, r)[0] for r in range(world)]


def choose_axis(ncells: int, nk: int, world: int) -> str:
    """What to split: cells when there are at least as many cells as ranks (config 4), else k-points."""
    return "cells" if ncells >= world and ncells > 1 else "kpoints"


def gather_shards(local, counts: Sequence[int], axis: int, group=None):
    """All-gather of the ranks' result blocks along ``axis`` (rank r contributed ``counts[r]`` slices), in rank order,
    which IS the original order because the ranges are contiguous.  ``local``: torch tensor (CUDA with an NCCL group, CPU
    with gloo).  Blocks are padded to the largest count so that one fixed-size collective serves ragged splits."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    if len(counts) != world or local.shape[axis] != counts[dist.get_rank(group)]:
        raise ValueError("gather_shards: counts do not match the group or the local block")
    moved = local.movedim(axis, 0).contiguous()
    cmax = max(counts)
    pad = torch.zeros((cmax,) + tuple(moved.shape[1:]), dtype=moved.dtype, device=moved.device)
    pad[: moved.shape[0]] = moved
    out = torch.empty((world * cmax,) + tuple(moved.shape[1:]), dtype=moved.dtype, device=moved.device)
    dist.all_gather_into_tensor(out, pad, group=group)
    parts = [out[r * cmax: r * cmax + counts[r]] for r in range(world)]
    return torch.cat(parts, dim=0).movedim(0, axis).contiguous()


def bands_sharded(cell_inputs, truncation: int, kpts, nbands: int, group=None, axis: str = "auto", device=None):
    """Whole band structure of ``cell_inputs`` (a list of (lattice, vert_offset, verts, compliance, density) tuples) on
    the ranks of ``group``: returns omega^2 as a torch tensor (ncells, nk, nbands), identical on every rank and bitwise
    equal to the single-rank result (each k-point's arithmetic does not depend on the batch it runs in).
    ``device``: torch device of this rank (default: current CUDA device)."""
    import torch
    import torch.distributed as dist
    from . import binding as bs

    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    k = np.ascontiguousarray(np.asarray(kpts, dtype=np.float64).reshape(-1, 2))
    ncells, nk = len(cell_inputs), k.shape[0]
    if axis == "auto":
        axis = choose_axis(ncells, nk, world)
    if device is None:
        device = torch.device("cuda", torch.cuda.current_device())
    if axis == "cells":
        lo, hi = shard_range(ncells, world, rank)
        mine, kl, counts, gaxis = list(cell_inputs[lo:hi]), k, shard_counts(ncells, world), 0
    elif axis == "kpoints":
        lo, hi = shard_range(nk, world, rank)
        mine, kl, counts, gaxis = list(cell_inputs), k[lo:hi], shard_counts(nk, world), 1
    else:
        raise ValueError("axis must be 'auto', 'cells' or 'kpoints'")
    local = torch.zeros((len(mine), kl.shape[0], nbands), dtype=torch.float64, device=device)
    if len(mine) and kl.shape[0]:
        cells = [bs.bs_create_cell(*ci) for ci in mine]
        for c in cells:
            bs.allocate_workspace(c, truncation, kl.shape[0], device=device)
        bs.bs_assemble_batch(cells, truncation)
        bs.bs_bands_batch(cells, kl, nbands, out=local)
        torch.cuda.synchronize(device)
        for c in cells:
            bs.bs_destroy_cell(c)
    if world == 1:
        return local
    backend = dist.get_backend(group)
    if backend == "nccl":
        return gather_shards(local, counts, gaxis, group)
    return gather_shards(local.cpu(), counts, gaxis, group).to(device)

"""Host-side sharding of target epochs over ranks (multi-GPU mode).

The batched mode fits many target epochs against one resident reference; epochs are independent
problems, so they shard over GPUs with no data-path collective: the reference is replicated, every
rank fits its own contiguous block of epochs, and only the fitted parameters are gathered at the end.
This module holds no device code and runs under any torch.distributed backend (tests use gloo).
"""
from __future__ import annotations

from typing import List, Tuple

import torch
import torch.distributed as dist


def epoch_shard(n_epochs: int, world_size: int, rank: int) -> Tuple[int, int]:
    """[start, stop) of the epochs owned by `rank`: contiguous blocks whose sizes differ by at most one,
    the first n_epochs % world_size ranks taking the larger blocks."""
    if world_size < 1 or not (0 <= rank < world_size) or n_epochs < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(n_epochs, world_size)
    start = rank * base + min(rank, extra)
    return start, start + base + (1 if rank < extra else 0)


def gather_epochs(local: torch.Tensor, n_epochs: int, group=None) -> torch.Tensor:
    """All-gathers per-epoch rows (e.g. fitted theta [E_local][np]) into [n_epochs][...] in epoch order.
    `local` must live where the backend can reach it (CPU for gloo, CUDA for nccl)."""
    world = dist.get_world_size(group)
    sizes = [epoch_shard(n_epochs, world, r) for r in range(world)]
    biggest = max(b - a for a, b in sizes)
    pad = torch.zeros((biggest,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    parts: List[torch.Tensor] = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    return torch.cat([parts[r][: b - a] for r, (a, b) in enumerate(sizes)], dim=0)


def max_over_ranks(value: float, device=None, group=None) -> float:
    """Maximum of a per-rank scalar (a device-measured duration) over all ranks."""
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


# ---- row bands of ONE image pair ------------------------------------------------------------
# The objective is a sum over valid pixels, so the valid rows split into bands: rank g evaluates the sub-image
# rows [r0, r1 + m - 1) of R and I -- whose own valid region is exactly the band -- with an ordinary handle, and the
# full loss and gradient are the sums of the per-rank results.  R is constant, so there is no halo exchange per
# evaluation; the only collective is one (m^2 + 2)-double all-gather, summed in rank order on every rank (deterministic,
# identical on all ranks).  Evaluation only: dia_fit's on-device loop has no place for a collective.
# Limits: (1) plain scalar background only -- with bg_degree > 0 every band's handle would centre and normalise the
# coordinates of Eq. 19 on its own sub-image, so the band sums would not add up to the full-image objective;
# (2) a flat field, mask or variance map must be sliced to the band's image rows by the caller, like R and I;
# (3) a rank whose band is empty (more ranks than valid rows) creates no handle and contributes zeros
# (`band_is_empty`; dia_create rejects an image smaller than the kernel).
def row_band(n_rows: int, m: int, world_size: int, rank: int) -> Tuple[int, int, int, int]:
    """-> (v0, v1, i0, i1): valid rows [v0, v1) owned by `rank` (indices into the valid region, n_rows - m + 1 rows in
    all, split like epoch_shard) and the image rows [i0, i1) = [v0, v1 + m - 1) to hand to dia_create / the targets."""
    n_valid = n_rows - m + 1
    if m < 1 or m % 2 == 0 or n_valid < 1:
        raise ValueError("bad image or kernel size")
    v0, v1 = epoch_shard(n_valid, world_size, rank)
    return v0, v1, v0, (v1 + m - 1 if v1 > v0 else v0)


def band_is_empty(band: Tuple[int, int, int, int]) -> bool:
    """True when row_band gave this rank no valid row: it must not call dia_create and contributes
    torch.zeros(m*m + 2, dtype=float64) to sum_over_ranks_in_order."""
    return band[1] <= band[0]


def sum_over_ranks_in_order(local: torch.Tensor, group=None) -> torch.Tensor:
    """All-gathers a small per-rank tensor (loss and gradient of a band, float64) and adds the parts in rank order on
    every rank: the same bits everywhere, whatever order the collective completes in."""
    world = dist.get_world_size(group)
    parts: List[torch.Tensor] = [torch.empty_like(local) for _ in range(world)]
    dist.all_gather(parts, local.contiguous(), group=group)
    total = torch.zeros_like(local)
    for r in range(world):
        total += parts[r]
    return total

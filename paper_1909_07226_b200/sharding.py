"""Host-side logic of the multi-GPU path: one process per GPU, the
baselines are sharded into contiguous ranges, every rank plans and grids its own range with no
data-path collective.  A caller that wants ONE grid sums the per-rank grids with a single
all-reduce after the adder (and broadcasts the model grid before the splitter).  Subgrids are
independent through gridder / subgrid FFT and inverse FFT / degridder (Alg. 1 / 2,
PAPER.md:283-306), so nothing else is exchanged.

Only torch.distributed plumbing lives here; no arithmetic of the method.
"""
from __future__ import annotations

from typing import Tuple

import torch
import torch.distributed as dist


def baseline_range(n_baselines: int, world_size: int, rank: int) -> Tuple[int, int]:
    """Contiguous, balanced range [begin, end) of baselines owned by `rank` (sizes differ by <= 1)."""
    if not (0 <= rank < world_size) or n_baselines < 0:
        raise ValueError("bad rank / world_size / n_baselines")
    base, extra = divmod(n_baselines, world_size)
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def shard_inputs(uvw: torch.Tensor, vis: torch.Tensor, baselines, world_size: int, rank: int):
    """Views of the rank's baselines: (uvw[b0:b1], vis[b0:b1], baselines[b0:b1], b0).  The A-terms,
    taper and frequencies are replicated."""
    b0, b1 = baseline_range(int(uvw.shape[0]), world_size, rank)
    return uvw[b0:b1].contiguous(), vis[b0:b1].contiguous(), baselines[b0:b1], b0


def allreduce_grid(grid: torch.Tensor, group=None) -> torch.Tensor:
    """Sum the per-rank [4][L][L] complex64 grids in place (viewed as float32: NCCL has no complex
    reduction).  One collective per gridding pass; a no-op without an initialised process group."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        flat = torch.view_as_real(grid) if grid.is_complex() else grid
        dist.all_reduce(flat, op=dist.ReduceOp.SUM, group=group)
    return grid


def broadcast_grid(grid: torch.Tensor, src: int = 0, group=None) -> torch.Tensor:
    """Model grid from `src` to every rank before the splitter (degridding direction)."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        flat = torch.view_as_real(grid) if grid.is_complex() else grid
        dist.broadcast(flat, src=src, group=group)
    return grid


def gather_visibilities(vis_local: torch.Tensor, n_baselines: int, group=None) -> torch.Tensor:
    """Concatenate the per-rank degridded visibilities [b0:b1][T][C][4] in rank order (ranges from
    baseline_range may differ in size by one, so this pads to the largest and trims)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return vis_local
    world = dist.get_world_size(group)
    sizes = [baseline_range(n_baselines, world, r) for r in range(world)]
    most = max(e - b for b, e in sizes)
    pad = torch.zeros((most,) + tuple(vis_local.shape[1:]), dtype=vis_local.dtype, device=vis_local.device)
    pad[: vis_local.shape[0]] = vis_local
    flat = torch.view_as_real(pad).contiguous()
    out = [torch.empty_like(flat) for _ in range(world)]
    dist.all_gather(out, flat, group=group)
    parts = [torch.view_as_complex(o)[: e - b] for o, (b, e) in zip(out, sizes)]
    return torch.cat(parts, dim=0)

"""Multi-GPU plumbing of the search.  One process per GPU.

The path has no exchange step ("each evaluation ... is entirely independent"): ranks
either search independent stacks (what bench.py --gpus N times) or disjoint bands of start rows of
one replicated stack.  The only collectives are the timing barrier / MAX reduction and, for
bands, the concatenation of the result planes.  Works with any torch.distributed backend (NCCL on
GPUs, gloo in the CPU tests); every function degrades to the single-process case.
"""
from __future__ import annotations

from typing import Callable, Dict, List, Optional, Tuple

import torch
import torch.distributed as dist


def world() -> Tuple[int, int]:
    """(rank, world_size); (0, 1) when torch.distributed is not initialised."""
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def rank_seed(seed: int, rank: int) -> int:
    """Seed of the independent synthetic stack a rank searches in the weak-scaling benchmark."""
    return int(seed) + 1000 * int(rank)


def row_bands(H: int, world_size: int) -> List[Tuple[int, int]]:
    """Balanced contiguous bands [y0, y1) of start rows, one per rank (empty if H < world_size)."""
    base, extra = divmod(int(H), int(world_size))
    out, y = [], 0
    for r in range(world_size):
        h = base + (1 if r < extra else 0)
        out.append((y, y + h))
        y += h
    return out


def max_over_ranks(value: float, device=None) -> float:
    """Device time of a step = the slowest rank's (MAX all-reduce); identity for one process."""
    _, n = world()
    if n == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def total_over_ranks(value: float, device=None) -> float:
    """Units processed by the whole job (SUM all-reduce)."""
    _, n = world()
    if n == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_bands(band: Dict[str, torch.Tensor], H: int) -> Dict[str, torch.Tensor]:
    """Concatenates per-rank result planes [rows_r, W, K] of row_bands(H, world) into [H, W, K] on
    every rank (all_gather of padded bands; no reduction: bands are disjoint)."""
    rank, n = world()
    if n == 1:
        return band
    bands = row_bands(H, n)
    hmax = max(y1 - y0 for y0, y1 in bands)
    out = {}
    for k, t in band.items():
        pad = torch.zeros((hmax,) + tuple(t.shape[1:]), dtype=t.dtype, device=t.device)
        pad[: t.shape[0]] = t
        parts = [torch.empty_like(pad) for _ in range(n)]
        dist.all_gather(parts, pad)
        out[k] = torch.cat([p[: y1 - y0] for p, (y0, y1) in zip(parts, bands)], 0)
    return out


def search_row_band(psiphi, times, vel_grid, K: int, min_obs: int, search: Optional[Callable] = None,
                    gather: bool = True, **kw) -> Dict[str, torch.Tensor]:
    """One stack, replicated on every rank, searched in start-row bands:
    this rank runs kbmod_search_rows on its band of row_bands(H, world) and, if `gather`, the bands
    are concatenated into [H, W, K] planes on every rank.  No collective on the data path of the
    search itself.  `search` defaults to binding.search (the C-ABI call); the CPU tests pass the
    same call of the SIMT-emulated library."""
    if search is None:
        from . import binding
        search = binding.search
    rank, n = world()
    H = int(psiphi.shape[1])
    y0, y1 = row_bands(H, n)[rank]
    band = search(psiphi, times, vel_grid, K, min_obs, y_begin=y0, y_end=y1, **kw)
    return gather_bands(band, H) if gather else band


def image_shares(N: int, world_size: int) -> List[Tuple[int, int]]:
    """Balanced contiguous shares [i0, i1) of the N images, one per rank (S2 sharded by image)."""
    return row_bands(N, world_size)


def make_psi_phi_sharded(sci: torch.Tensor, var: torch.Tensor, mask: Optional[torch.Tensor], psf,
                         make: Optional[Callable] = None) -> torch.Tensor:
    """S1+S2 of ONE stack on all ranks: rank r builds psi/phi of its share of
    the images (kbmod_make_psi_phi on a slice of the stack) and ONE all-gather (NCCL over NVLink on
    GPUs, gloo in the CPU tests) replicates the float2 stack on every rank, ready for the row-band
    search.  This is the only exchange step of the multi-GPU path; images are independent, so the
    gathered stack is bit-identical to a single-rank build.  `make` defaults to binding.make_psi_phi."""
    if make is None:
        from . import binding
        make = binding.make_psi_phi
    rank, n = world()
    N, H, W = sci.shape
    if n == 1:
        return make(sci, var, mask, psf)
    shares = image_shares(N, n)
    i0, i1 = shares[rank]
    cmax = max(b - a for a, b in shares)
    part = torch.zeros((cmax, H, W, 2), dtype=torch.float32, device=sci.device)
    if i1 > i0:
        part[: i1 - i0] = make(sci[i0:i1].contiguous(), var[i0:i1].contiguous(),
                               None if mask is None else mask[i0:i1].contiguous(), psf[i0:i1])
    parts = [torch.empty_like(part) for _ in range(n)]
    dist.all_gather(parts, part)
    return torch.cat([p[: b - a] for p, (a, b) in zip(parts, shares)], 0).contiguous()

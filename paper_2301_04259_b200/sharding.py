"""Multi-GPU plumbing: one process per GPU, independent units per rank, no data-path collective.

The path shards without an exchange step: stars are independent, phases are independent
given the spectra, and wavelength slices need only a read-only halo.  The units of a job (stars of a sweep,
or phases of one star) are dealt to the ranks in contiguous blocks; every rank runs the same C-ABI calls on
its block and nothing crosses NVLink while it computes.  The only communication is bookkeeping: the
max-over-ranks of a device-side duration (bench.py) and, optionally, gathering small per-unit summaries.
Works with the `nccl` backend on GPUs and with `gloo` on CPU (tests/test_sharding_gloo.py).
"""
from __future__ import annotations

from typing import List, Sequence, Tuple

import torch
import torch.distributed as dist


def shard_range(n_units: int, rank: int, world: int) -> Tuple[int, int]:
    """[begin, end) of the units rank `rank` owns when n_units are dealt to `world` ranks in contiguous blocks
    whose sizes differ by at most one (the first n_units % world ranks get the larger block)."""
    if world < 1 or not 0 <= rank < world or n_units < 0:
        raise ValueError("bad shard request")
    base, extra = divmod(n_units, world)
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def shard_list(units: Sequence, rank: int, world: int) -> list:
    b, e = shard_range(len(units), rank, world)
    return list(units[b:e])


def world_info() -> Tuple[int, int]:
    """(rank, world) of the initialised process group, or (0, 1) without one."""
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def max_over_ranks(value: float, device=None) -> float:
    """Max of a per-rank scalar (a device-timed duration) over all ranks; the value itself when not distributed."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_unit_summaries(local: torch.Tensor, n_units: int) -> torch.Tensor:
    """All ranks' per-unit summary rows (e.g. one checksum per star), in unit order, on every rank.

    `local` holds this rank's rows [n_local, k] for the block shard_range gives it.  Blocks differ in length by
    at most one, so rows are padded to the longest block for the all_gather and trimmed afterwards."""
    rank, world = world_info()
    if world == 1:
        return local
    longest = (n_units + world - 1) // world
    pad = torch.zeros((longest,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    parts: List[torch.Tensor] = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    rows = []
    for r in range(world):
        b, e = shard_range(n_units, r, world)
        rows.append(parts[r][: e - b])
    return torch.cat(rows, dim=0)

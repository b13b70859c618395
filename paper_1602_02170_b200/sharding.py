"""Sharding of the mobility matvec across ranks (one process per GPU).

Two ways to split u = M lambda over G GPUs, both with every rank holding all positions and forces:

* rows (this module's ``shard_rows`` + ``gather_velocities``): rank r computes its slice of target
  rows against all sources, then one all-gather.  Needs the plain kernel (every ordered pair).
* work (``rpy_*_matvec_shard`` + ``reduce_velocities``): rank r computes 1/G of the UNORDERED tile
  pairs with the symmetric kernel (M_ij = M_ji^T) and so contributes to every row;
  one all-reduce (sum) of the 3 k N partial velocities gives u on every rank.  Per-GPU arithmetic
  is 33 instead of 56 FP-pipe operations per ordered pair, at the price of 2x the bytes on NVLink
  (still O(N) against O(N^2 / G) arithmetic).

Row sharding, in detail:

Rows of M are independent ("trivially parallelized"): rank r computes the
velocities of a contiguous slice of target blobs against ALL source blobs with
``rpy_wall_matvec(..., rows=shard_rows(n, r, world))`` and needs no communication to do so.
Only a caller that wants the whole ``u`` on every rank (a Krylov iteration) exchanges data:
one all-gather of ``3 k N`` elements, ``gather_velocities`` below.

Host logic only: no arithmetic of the method lives here.  It works with any
``torch.distributed`` backend (NCCL on the GPUs; gloo in the CPU test).
"""
from __future__ import annotations

from typing import List, Optional, Tuple

import torch


def row_partition(n_blobs: int, world: int) -> List[Tuple[int, int]]:
    """``[(row_begin, row_count)] * world``: contiguous, ordered, covering ``0..n_blobs-1``,
    sizes differing by at most one (rank r gets rows ``r*n//world .. (r+1)*n//world - 1``)."""
    if n_blobs < 0 or world < 1:
        raise ValueError("row_partition: n_blobs >= 0 and world >= 1 required")
    bounds = [r * n_blobs // world for r in range(world + 1)]
    return [(bounds[r], bounds[r + 1] - bounds[r]) for r in range(world)]


def shard_rows(n_blobs: int, rank: int, world: int) -> Tuple[int, int]:
    """The ``rows=(row_begin, row_count)`` argument of the matvec calls for ``rank``."""
    if not 0 <= rank < world:
        raise ValueError("shard_rows: 0 <= rank < world required")
    return row_partition(n_blobs, world)[rank]


def gather_buffers(n_blobs: int, n_rhs: int, world: int, dtype, device) -> List[torch.Tensor]:
    """Receive buffers for ``gather_velocities`` (allocate once, reuse).  All have the size of
    the largest shard, ``[k, ceil(n/world), 3]``: equal-sized buffers work with every backend."""
    cmax = max(c for _, c in row_partition(n_blobs, world))
    return [torch.empty((n_rhs, cmax, 3), dtype=dtype, device=device) for _ in range(world)]


def gather_velocities(local: torch.Tensor, n_blobs: int, group=None,
                      buffers: Optional[List[torch.Tensor]] = None,
                      concatenate: bool = True):
    """All-gather the per-rank velocity slices ``[k, row_count_r, 3]`` (slice sizes may differ by
    one; shorter slices travel padded by one row) and, if ``concatenate``, return the full
    ``[k, n_blobs, 3]`` tensor in blob order on every rank; otherwise the list of slices (views)."""
    import torch.distributed as dist
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    if local.dim() != 3 or local.shape[2] != 3:
        raise ValueError("gather_velocities: local must be [k, rows, 3]")
    part = row_partition(n_blobs, world)
    if local.shape[1] != part[rank][1]:
        raise ValueError(f"gather_velocities: rank {rank} holds {local.shape[1]} rows, its shard has {part[rank][1]}")
    if buffers is None:
        buffers = gather_buffers(n_blobs, local.shape[0], world, local.dtype, local.device)
    cmax = buffers[0].shape[1]
    if local.shape[1] == cmax:
        send = local.contiguous()
    else:
        send = torch.zeros_like(buffers[rank])     # shorter shard: pad by one row
        send[:, :local.shape[1]].copy_(local)
    dist.all_gather(buffers, send, group=group)
    slices = [buffers[r][:, :part[r][1]] for r in range(world)]
    if not concatenate:
        return slices
    return torch.cat(slices, dim=1)


def reduce_velocities(partial: torch.Tensor, group=None) -> torch.Tensor:
    """Sum the per-rank PARTIAL velocities of ``rpy_*_matvec_shard`` (full length on every rank, float64
    on both precision paths so that the cross-rank sum stays an fp64 accumulation) in place with one
    all-reduce; returns ``partial``, which then holds u on every rank."""
    import torch.distributed as dist
    if partial.dtype != torch.float64:
        raise TypeError("reduce_velocities: the partial products of rpy_*_matvec_shard are float64")
    dist.all_reduce(partial, op=dist.ReduceOp.SUM, group=group)
    return partial


class _DevicePointer:
    """Lets torch wrap `count` float64 values at a raw device address (CUDA array interface, version 2)."""

    def __init__(self, ptr: int, count: int):
        self.__cuda_array_interface__ = {"shape": (count,), "typestr": "<f8", "data": (ptr, False), "version": 2}


def wrap_doubles(ptr: int, count: int, device=None) -> torch.Tensor:
    """A float64 tensor VIEW of `count` doubles at address `ptr`: device memory when `device` is a CUDA device,
    else host memory.  No copy; the caller keeps the memory alive."""
    if device is not None and torch.device(device).type == "cuda":
        return torch.as_tensor(_DevicePointer(ptr, count), device=device)
    import ctypes
    import numpy as np
    buf = (ctypes.c_double * count).from_address(ptr)
    return torch.from_numpy(np.frombuffer(buf, dtype=np.float64, count=count))


def solve_reduce_hook(group=None, device=None):
    """The `reduce(ptr, count)` hook of a multi-GPU ``rpy_rigid_mobility_solve(..., shard, n_shards, reduce)``:
    one in-place all-reduce (sum) per product over the ranks' partial velocities, ordered on the current
    stream like every torch.distributed collective.  Every rank runs the same replicated Krylov process on
    the summed product, so all ranks take the same decisions and return the same solution."""
    import torch.distributed as dist

    def reduce(ptr: int, count: int):
        dist.all_reduce(wrap_doubles(ptr, count, device), op=dist.ReduceOp.SUM, group=group)
    return reduce

"""Datapoint-sharded FK convolution over several GPUs: one process per GPU.

Rows of an FK table are independent (Eq. (1): one sigma^N per datapoint N), so a table -- or the
whole tables of a ragged group -- is split over the ranks by datapoints; `f` (<= 0.7 MB) is replicated.

  forward   no exchange: every rank holds its slice sigma[n0:n1][R]; `gather_sigma` collects the slices when one
            place needs them all (all_gather of padded slices; the padding is dropped);
  VJP       every rank produces a partial df[R][nfl][nx] over its datapoints; ONE all-reduce(sum) completes it
            (NCCL over NVLink on GPUs, gloo in the CPU tests).  The sum order then depends on the world size,
            so results are bitwise repeatable per world size, not across world sizes.

This module holds the host-side plan and the two collectives; the arithmetic is the C-ABI library's
(`fkconv.FkTable`).  Nothing here imports `oracle/`.
"""
from __future__ import annotations

from typing import List, Sequence, Tuple

import numpy as np
import torch
import torch.distributed as dist


def shard_rows(N: int, world: int, rank: int) -> Tuple[int, int]:
    """Contiguous, balanced datapoint range [n0, n1) of `rank` (sizes differ by at most one)."""
    if N < 0 or world <= 0 or not 0 <= rank < world:
        raise ValueError("shard_rows: bad arguments")
    return N * rank // world, N * (rank + 1) // world


def shard_tables(cost: Sequence[float], world: int) -> List[List[int]]:
    """Whole tables to ranks, balanced by cost (bytes of FK): longest-processing-time greedy, ties by index.
    Returns, per rank, the table indices in ascending order.  Deterministic."""
    if world <= 0:
        raise ValueError("shard_tables: world <= 0")
    order = sorted(range(len(cost)), key=lambda t: (-float(cost[t]), t))
    load = [0.0] * world
    out: List[List[int]] = [[] for _ in range(world)]
    for t in order:
        r = min(range(world), key=lambda q: (load[q], q))
        out[r].append(t)
        load[r] += float(cost[t])
    return [sorted(x) for x in out]


def _world(group=None) -> Tuple[int, int]:
    if dist.is_available() and dist.is_initialized():
        return dist.get_world_size(group), dist.get_rank(group)
    return 1, 0


def allreduce_df(df_partial: torch.Tensor, group=None) -> torch.Tensor:
    """Completes the VJP: sum over ranks of the per-rank partial df (in place).  The one data-path collective."""
    world, _ = _world(group)
    if world > 1:
        dist.all_reduce(df_partial, op=dist.ReduceOp.SUM, group=group)
    return df_partial


def gather_sigma(sigma_local: torch.Tensor, N: int, group=None) -> torch.Tensor:
    """sigma[N][R] on every rank from the rank-local slices of `shard_rows` (optional: the forward needs no exchange)."""
    world, rank = _world(group)
    if world == 1:
        return sigma_local
    R = sigma_local.shape[1]
    rows = max(shard_rows(N, world, r)[1] - shard_rows(N, world, r)[0] for r in range(world))
    pad = torch.zeros((rows, R), dtype=sigma_local.dtype, device=sigma_local.device)
    pad[: sigma_local.shape[0]] = sigma_local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    out = torch.empty((N, R), dtype=sigma_local.dtype, device=sigma_local.device)
    for r in range(world):
        n0, n1 = shard_rows(N, world, r)
        out[n0:n1] = parts[r][: n1 - n0]
    return out


class ShardedFkTable:
    """One table split by datapoints over the ranks of `group`; each rank keeps (and packs) only its rows."""

    def __init__(self, kind, fk_logical_host: np.ndarray, index_list, nfl, group=None, device=None, **kw):
        from . import fkconv  # fails loudly without the CUDA library: there is no CPU fallback
        self.group = group
        self.world, self.rank = _world(group)
        self.N = int(fk_logical_host.shape[0])
        self.n0, self.n1 = shard_rows(self.N, self.world, self.rank)
        if self.n1 <= self.n0:
            raise ValueError("ShardedFkTable: more ranks than datapoints")
        dev = torch.device("cuda", torch.cuda.current_device()) if device is None else device
        local = torch.from_numpy(np.ascontiguousarray(fk_logical_host[self.n0:self.n1])).to(dev)
        self.table = fkconv.FkTable(kind, local, index_list, nfl, **kw)

    def conv(self, f, stream=None):
        """Local slice sigma[n0:n1][R] (no communication)."""
        return self.table.conv(f, stream=stream)

    def conv_all(self, f, stream=None):
        return gather_sigma(self.conv(f, stream=stream), self.N, self.group)

    def vjp(self, f, g_local, stream=None):
        """g_local = g[n0:n1][R]; returns the complete df[R][nfl][nx] on every rank (one all-reduce)."""
        return allreduce_df(self.table.vjp(f, g_local, stream=stream), self.group)

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


class _on_stream:
    """Runs the collective on the stream the local kernels were launched on.  NCCL orders a collective against
    torch's CURRENT stream: if the kernels went to another stream, the all-reduce could read df before they wrote
    it.  No-op on CPU tensors (gloo in the tests) and when no stream was given."""

    def __init__(self, t: torch.Tensor, stream):
        self.ctx = None
        if stream is not None and t.is_cuda:
            st = stream if isinstance(stream, torch.cuda.Stream) else torch.cuda.ExternalStream(int(stream))
            self.ctx = torch.cuda.stream(st)

    def __enter__(self):
        if self.ctx is not None:
            self.ctx.__enter__()

    def __exit__(self, *a):
        if self.ctx is not None:
            self.ctx.__exit__(*a)


def allreduce_df(df_partial: torch.Tensor, group=None, stream=None) -> torch.Tensor:
    """Completes the VJP: sum over ranks of the per-rank partial df (in place).  The one data-path collective."""
    world, _ = _world(group)
    if world > 1:
        with _on_stream(df_partial, stream):
            dist.all_reduce(df_partial, op=dist.ReduceOp.SUM, group=group)
    return df_partial


def gather_sigma(sigma_local: torch.Tensor, N: int, group=None, stream=None) -> torch.Tensor:
    """sigma[N][R] on every rank from the rank-local slices of `shard_rows` (optional: the forward needs no exchange)."""
    world, rank = _world(group)
    if world == 1:
        return sigma_local
    R = sigma_local.shape[1]
    rows = max(shard_rows(N, world, r)[1] - shard_rows(N, world, r)[0] for r in range(world))
    with _on_stream(sigma_local, stream):
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
        return gather_sigma(self.conv(f, stream=stream), self.N, self.group, stream)

    def vjp(self, f, g_local, stream=None):
        """g_local = g[n0:n1][R]; returns the complete df[R][nfl][nx] on every rank (one all-reduce)."""
        return allreduce_df(self.table.vjp(f, g_local, stream=stream), self.group, stream)


# ------------------------------------------------------------------------------------------------ ragged group
class GroupPlan:
    """Whole tables of a ragged group to ranks ("whole tables of a ragged group, balanced by bytes").

    `shapes` = per table (N, nx, nfl, C); the cost of a table is its FK bytes N * C * nx^2.  Holds, for R
    replicas, the element offsets of every table inside the GLOBAL concatenations f_cat / df_cat
    (sum_t R*nfl_t*nx_t) and sigma_cat / g_cat (sum_t N_t*R) -- the layout of fk_group_offsets over all tables --
    and which tables each rank owns."""

    def __init__(self, shapes: Sequence[Tuple[int, int, int, int]], world: int):
        self.shapes = [tuple(int(v) for v in s) for s in shapes]
        self.world = world
        self.owner_tables = shard_tables([N * C * nx * nx for (N, nx, nfl, C) in self.shapes], world)
        self.owner = [0] * len(self.shapes)
        for r, ts in enumerate(self.owner_tables):
            for t in ts:
                self.owner[t] = r

    def offsets(self, R: int):
        fo, so = [0], [0]
        for (N, nx, nfl, C) in self.shapes:
            fo.append(fo[-1] + R * nfl * nx)
            so.append(so[-1] + N * R)
        return fo, so

    def scatter_local(self, pieces: Sequence[torch.Tensor], rank: int, offs: Sequence[int]) -> torch.Tensor:
        """Zero-filled global concatenation with this rank's per-table pieces (ascending table order) in place."""
        dev, dt = (pieces[0].device, pieces[0].dtype) if len(pieces) else (torch.device("cpu"), torch.float64)
        out = torch.zeros(int(offs[-1]), dtype=dt, device=dev)
        for t, p in zip(self.owner_tables[rank], pieces):
            out[offs[t]:offs[t + 1]] = p.reshape(-1)
        return out


def allreduce_cat(cat_local: torch.Tensor, group=None, stream=None) -> torch.Tensor:
    """Every table's slice is non-zero on exactly one rank, so the sum is an exact assembly: x + 0 = x, the result
    is bit-identical to the unsharded concatenation whatever the world size."""
    return allreduce_df(cat_local, group, stream)


class ShardedFkGroup:
    """A ragged group with whole tables owned by ranks (`GroupPlan`); each rank packs only its tables into an
    `fkconv.FkGroup`.  `f_cat` (global layout, <= a few MB) is replicated; forward: no exchange, the local
    sigma pieces are assembled on demand; VJP: df is per table (reading R14), the global df_cat is assembled by
    the one all-reduce."""

    def __init__(self, cases, group=None, device=None, R_hint=1, **kw):
        """cases[t] = (kind, fk_logical_host, index_list, nfl) for EVERY table; only the owned ones are uploaded."""
        from . import fkconv
        self.K = fkconv
        self.group = group
        self.world, self.rank = _world(group)
        shapes = []
        for (kind, fk, idx, nfl) in cases:
            N, nx, C = int(fk.shape[0]), int(fk.shape[1]), int(fk.shape[-1])
            shapes.append((N, nx, nfl, C))
        self.plan = GroupPlan(shapes, self.world)
        self.mine = self.plan.owner_tables[self.rank]
        if not self.mine:
            raise ValueError("ShardedFkGroup: more ranks than tables")
        dev = torch.device("cuda", torch.cuda.current_device()) if device is None else device
        self.tables = []
        for t in self.mine:
            kind, fk, idx, nfl = cases[t]
            self.tables.append(fkconv.FkTable(kind, torch.from_numpy(np.ascontiguousarray(fk)).to(dev), idx, nfl, **kw))
        self.local = fkconv.FkGroup(self.tables, R_hint=R_hint)

    def _local_cat(self, cat: torch.Tensor, offs) -> torch.Tensor:
        return torch.cat([cat[offs[t]:offs[t + 1]] for t in self.mine])

    def conv(self, f_cat, R, stream=None):
        """Local sigma pieces (concatenated over the owned tables, ascending); no communication."""
        fo, _ = self.plan.offsets(R)
        return self.local.conv(self._local_cat(f_cat, fo), R, stream=stream)

    def conv_all(self, f_cat, R, stream=None):
        _, so = self.plan.offsets(R)
        loc = self.conv(f_cat, R, stream)
        lo = np.cumsum([0] + [so[t + 1] - so[t] for t in self.mine])
        pieces = [loc[lo[k]:lo[k + 1]] for k in range(len(self.mine))]
        return allreduce_cat(self.plan.scatter_local(pieces, self.rank, so), self.group, stream)

    def vjp(self, f_cat, g_cat, R, stream=None):
        """g_cat in the global layout; returns the complete df_cat (global layout) on every rank."""
        fo, so = self.plan.offsets(R)
        loc = self.local.vjp(self._local_cat(f_cat, fo), self._local_cat(g_cat, so), R, stream=stream)
        lo = np.cumsum([0] + [fo[t + 1] - fo[t] for t in self.mine])
        pieces = [loc[lo[k]:lo[k + 1]] for k in range(len(self.mine))]
        return allreduce_cat(self.plan.scatter_local(pieces, self.rank, fo), self.group, stream)

    def destroy(self):
        self.local.destroy()
        for t in self.tables:
            t.destroy()

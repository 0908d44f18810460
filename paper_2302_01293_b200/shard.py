"""Shard-by-star multi-GPU plumbing (host logic only: every quantity of the search
is "determined for each star", so stars are independent units and the path has no exchange step).

  * :func:`lpt_partition` -- stars are dealt to ranks by cost N_pts x n_freq with the longest-processing-time
    greedy rule (the top 1 % of a production-shaped batch holds ~20 % of the work, so equal counts do not balance);
  * :func:`gather_tables` -- the one collective of a job: every rank's per-star result table (peaks, statistics,
    ...; fixed-size records) goes to all ranks with ONE ``all_gather`` over ``torch.distributed`` (NCCL on GPUs,
    gloo in the CPU tests) and is put back into global star order.

Nothing here touches the search arithmetic; the kernels never communicate.
"""
from __future__ import annotations

import heapq

import numpy as np


def lpt_partition(cost, world: int):
    """Longest-processing-time greedy: stars in order of decreasing cost (ties: lower index first), each to the
    rank with the least load so far (ties: lower rank).  Deterministic, so every rank computes the same answer
    from the same costs.  -> list of ``world`` sorted int64 index arrays (a partition of range(len(cost)))."""
    cost = np.asarray(cost, dtype=np.float64)
    if world < 1:
        raise ValueError("world must be >= 1")
    order = np.lexsort((np.arange(cost.size), -cost))
    heap = [(0.0, r) for r in range(world)]
    heapq.heapify(heap)
    parts = [[] for _ in range(world)]
    for i in order:
        load, r = heapq.heappop(heap)
        parts[r].append(int(i))
        heapq.heappush(heap, (load + float(cost[i]), r))
    return [np.array(sorted(p), dtype=np.int64) for p in parts]


def imbalance(cost, parts) -> float:
    """max over ranks of the summed cost / mean over ranks (1.0 = perfectly balanced)."""
    cost = np.asarray(cost, dtype=np.float64)
    loads = np.array([cost[p].sum() for p in parts])
    return float(loads.max() / loads.mean()) if loads.mean() > 0 else 1.0


def pack_rows(local_table, local_ids):
    """[S_local, ...] records + global ids -> uint8 [S_local, rec] rows of (valid flag, global id, record bytes)."""
    local_table = np.ascontiguousarray(local_table)
    local_ids = np.ascontiguousarray(local_ids, dtype=np.int64)
    if local_table.shape[0] != local_ids.size:
        raise ValueError("one row of the table per local star id")
    row_bytes = int(np.prod(local_table.shape[1:], dtype=np.int64)) * local_table.dtype.itemsize
    rec = 16 + row_bytes
    rec += (-rec) % 8
    buf = np.zeros((local_ids.size, rec), dtype=np.uint8)
    if local_ids.size:
        buf[:, 0:8] = np.ones(local_ids.size, dtype=np.int64).view(np.uint8).reshape(-1, 8)
        buf[:, 8:16] = local_ids.view(np.uint8).reshape(-1, 8)
        buf[:, 16:16 + row_bytes] = local_table.view(np.uint8).reshape(local_ids.size, row_bytes)
    return buf


def unpack_rows(all_rows, n_global: int, dtype, row_shape=()):
    """uint8 [n, rec] rows from every rank (padding rows have flag 0) -> table [n_global, ...] in global order."""
    dtype = np.dtype(dtype)
    row_shape = tuple(row_shape)
    row_bytes = int(np.prod(row_shape, dtype=np.int64)) * dtype.itemsize
    allb = np.ascontiguousarray(all_rows).reshape(-1, all_rows.shape[-1])
    valid = allb[:, 0:8].copy().view(np.int64).ravel() == 1
    ids = allb[:, 8:16].copy().view(np.int64).ravel()[valid]
    if ids.size != n_global or np.unique(ids).size != n_global or (ids.size and (ids.min() < 0 or ids.max() >= n_global)):
        raise RuntimeError(f"unpack_rows: {ids.size} rows for {n_global} stars (shards do not partition the job)")
    out = np.zeros((n_global,) + row_shape, dtype=dtype)
    out[ids] = np.ascontiguousarray(allb[valid, 16:16 + row_bytes]).view(dtype).reshape((ids.size,) + row_shape)
    return out


def max_rows_over_ranks(n_local: int, device=None) -> int:
    """Largest shard size of the job (shards differ under LPT): the padded row count of the gather."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return int(n_local)
    n = torch.tensor([n_local], dtype=torch.int64, device=torch.device(device) if device is not None else "cpu")
    dist.all_reduce(n, op=dist.ReduceOp.MAX)
    return int(n.item())


def gather_rows(rows, n_max: int, out=None):
    """ONE all_gather of fixed-size rows: torch uint8 [S_local, rec] (zero-padded to n_max rows) from every rank
    -> torch uint8 [world, n_max, rec] on the same device.  NCCL for CUDA tensors, gloo for CPU tensors."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size() if (dist.is_available() and dist.is_initialized()) else 1
    rec = rows.shape[1]
    send = rows
    if rows.shape[0] != n_max:
        send = torch.zeros((n_max, rec), dtype=torch.uint8, device=rows.device)
        send[:rows.shape[0]] = rows
    if out is None:
        out = torch.empty((world, n_max, rec), dtype=torch.uint8, device=rows.device)
    if world == 1:
        out[0].copy_(send)
    else:
        # the one data collective of a job (output in its concatenated [world * n_max, rec] form: NCCL and gloo both take it)
        dist.all_gather_into_tensor(out.view(world * n_max, rec), send.contiguous())
    return out


def gather_tables(local_table, local_ids, n_global: int, device=None):
    """All ranks' per-star tables in global star order, by ONE all_gather.

    ``local_table``: numpy array [S_local, ...] of fixed-size records (any dtype, e.g. the structured peak table
    [S_local, top_k]); ``local_ids``: int64[S_local] global star index of each row; ``n_global``: total number of
    stars of the job.  Every rank gets the full table [n_global, ...] (rank 0 is the one that reports it).
    Rows are padded to the largest shard so that a single fixed-size all_gather moves ids and records together.
    Without an initialised process group (one GPU) the local table is just put in order.
    """
    import torch
    local_table = np.ascontiguousarray(local_table)
    rows = torch.from_numpy(pack_rows(local_table, local_ids))
    if device is not None:
        rows = rows.to(torch.device(device))
    n_max = max_rows_over_ranks(rows.shape[0], device)
    allr = gather_rows(rows, n_max).cpu().numpy()
    return unpack_rows(allr, n_global, local_table.dtype, local_table.shape[1:])

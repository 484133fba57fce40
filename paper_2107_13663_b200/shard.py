"""Marker sharding across ranks: independent shards, no data-path collective.

Markers are independent and the paper runs every GPU with the whole field table and no traffic during
the push, so rank r of N simply owns its own shard of markers.  This module holds the bookkeeping that
``bench.py`` uses under torchrun: the per-rank seed, the per-rank slice of a global id range, and the reduction of the
per-rank timings to the whole-job figure (max over ranks).  No arithmetic of the method lives here.
"""
from __future__ import annotations

from typing import Sequence, Tuple


def shard_seed(config: int, rank: int) -> int:
    """Seed of rank's shard: rank 0 draws the documented seed 1000 + config."""
    return 1000 + int(config) + 7919 * int(rank)


def shard_range(n_global: int, rank: int, world: int) -> Tuple[int, int]:
    """[begin, end) of the global marker ids owned by `rank` when n_global markers are split over `world` ranks
    (contiguous blocks, the first n_global % world ranks get one more)."""
    if world < 1 or not 0 <= rank < world or n_global < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(int(n_global), int(world))
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def whole_job_rate(markers_per_rank: Sequence[int], steps: int, ms_max_over_ranks: float) -> float:
    """particle-steps/s of the whole job: all markers of all ranks x steps / the slowest rank's device time."""
    return float(sum(int(m) for m in markers_per_rank)) * steps / (ms_max_over_ranks * 1e-3)


def max_over_ranks(values, dist=None, device=None):
    """Element-wise maximum of a list of floats over the ranks of torch.distributed (identity without a group)."""
    import torch

    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist is not None and dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


# ---- the two exchange steps around the push ----------------------------------------------
# (1) the field image goes from the rank that built it to every other rank once per field update; (2) the deposited
# moments of the marker shards are summed.  Both are plain collectives on whole buffers (NCCL on device tensors, gloo on
# CPU tensors in the tests); the push itself exchanges nothing.

def broadcast_bytes(buf, dist, src: int = 0):
    """Broadcast a uint8 tensor whose length only `src` knows.  `buf` is the tensor on `src` and None (or anything) on the
    other ranks, which get a fresh tensor on `like_device`.  Returns the tensor every rank now holds."""
    import torch

    rank = dist.get_rank()
    dev = buf.device if rank == src else None
    n = torch.tensor([buf.numel() if rank == src else 0], dtype=torch.int64)
    backend = dist.get_backend()
    if backend == "nccl":
        n = n.cuda()
    dist.broadcast(n, src)
    if rank != src:
        dev = torch.device("cuda", torch.cuda.current_device()) if backend == "nccl" else torch.device("cpu")
        buf = torch.empty(int(n.item()), dtype=torch.uint8, device=dev)
    dist.broadcast(buf, src)
    return buf


def broadcast_fields(pusher, dist, n_elems: int, n_modes: int, src: int = 0):
    """"the fields ... are collected and uploaded to every GPU".  Rank `src` has called fields_create; its
    self-describing fields workspace is broadcast and every other rank binds its copy with m3dk_fields_attach (no host
    tables, no second least-squares fit or search-grid build)."""
    ws = broadcast_bytes(pusher.fields_workspace() if dist.get_rank() == src else None, dist, src)
    if dist.get_rank() != src:
        pusher.fields_attach(ws, n_elems, n_modes)
    return ws.numel()


def allreduce_moments(rhs, dist):
    """Sum of the deposited moment tables of all marker shards, in place on every rank."""
    if dist is not None and dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(rhs, op=dist.ReduceOp.SUM)
    return rhs

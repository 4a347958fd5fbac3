"""Multi-GPU plumbing for the replica scheme.

The path shards by input: every rank owns a private filter replica and a contiguous slice of the
insert batch (k-mer start positions, or whole records); after the local inserts ONE exchange step
makes the replicas identical — a bitwise-OR all-reduce of the filter bytes.  NCCL has no OR
reduction, so it is an all-gather of (a window of) the replicas followed by the library's
``sbf_or_bits_device`` kernel.  Queries then shard by reads with no collective at all.

Only argument marshalling and ``torch.distributed`` calls live here; nothing of the filter's
arithmetic.  The partition helpers are pure functions so that world_size-2 gloo tests can check
them on CPU.
"""
from __future__ import annotations

from typing import Callable, List, Tuple

import numpy as np


def partition_positions(total: int, k: int, world: int, rank: int) -> Tuple[int, int]:
    """Byte range [a, e) of one sequence that rank must see so that every k-mer START position
    in [a, a + share) is complete inside it: shares are equal slices of the start positions and
    each range is extended by the k-1 symbol halo (P:151 uses the same halo per tile)."""
    if total <= 0:
        return 0, 0
    n_start = max(total - k + 1, 0)          # k-mer start positions of the whole sequence
    if n_start == 0:
        return (0, total) if rank == 0 else (0, 0)
    per = -(-n_start // world)
    a = min(rank * per, n_start)
    b = min(a + per, n_start)
    if a == b:
        return a, a
    return a, b + k - 1


def partition_records(offsets: np.ndarray, world: int, rank: int) -> Tuple[int, int]:
    """Contiguous record range [r0, r1) for rank, balanced by symbols (records are never split:
    no k-mer spans two records, so there is no halo)."""
    off = np.asarray(offsets, dtype=np.uint64)
    n_rec = off.size - 1
    if n_rec <= 0:
        return 0, 0
    total = int(off[-1])
    # the r-th cut is the first record boundary at or after r * total / world
    cuts = [int(np.searchsorted(off, np.uint64((total * r) // world), side="left")) for r in range(world + 1)]
    cuts[0], cuts[-1] = 0, n_rec
    for i in range(1, world + 1):
        cuts[i] = max(cuts[i], cuts[i - 1])
    return cuts[rank], cuts[rank + 1]


def rebase_offsets(offsets: np.ndarray, r0: int, r1: int) -> np.ndarray:
    """offsets[r0..r1] shifted to start at 0 (what sbf_*_records wants for a slice of a batch)."""
    off = np.asarray(offsets, dtype=np.uint64)
    return (off[r0:r1 + 1] - off[r0]).astype(np.uint64)


def or_allreduce(local, or_into: Callable[[object], None], group=None, window_bytes: int = 1 << 28) -> int:
    """Make every rank's replica the OR of all replicas.

    local    : 1-D uint8 torch tensor viewing this rank's replica (device tensor under NCCL,
               CPU tensor under gloo); read during the gathers, updated by ``or_into``.
    or_into  : callable(offset_bytes, peer_chunk_tensor) that ORs a peer's chunk into the local
               replica at that byte offset (sbf_or_bits_device on a sub-range for the GPU path).
    The replicas are exchanged window by window so the gather buffer stays at
    world * window_bytes (a 4 GiB filter on 8 ranks would otherwise need 32 GiB of scratch).
    Returns the number of OR calls issued.
    """
    import torch
    import torch.distributed as dist

    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    if world == 1:
        return 0
    n = local.numel()
    window = min(n, max(32, window_bytes - window_bytes % 32))
    gathered = torch.empty(world * window, dtype=torch.uint8, device=local.device)
    calls = 0
    for a in range(0, n, window):
        w = min(window, n - a)
        outs: List = [gathered[r * window:r * window + w] for r in range(world)]
        dist.all_gather(outs, local[a:a + w].contiguous(), group=group)
        for r in range(world):
            if r != rank:
                or_into(a, outs[r])
                calls += 1
    return calls


class DevicePtrView:
    """Exposes a raw device pointer to torch (``torch.as_tensor(view, device='cuda')``) through the
    CUDA array interface — used to hand the library-owned filter to torch.distributed."""

    def __init__(self, ptr: int, nbytes: int):
        self.__cuda_array_interface__ = {
            "shape": (nbytes,), "typestr": "|u1", "data": (ptr, False), "version": 3, "strides": None,
        }


def filter_tensor(handle):
    """The library-owned filter replica as a uint8 CUDA tensor (no copy)."""
    import torch
    from . import sbf_filter_device_ptr, sbf_num_shards
    n = sbf_num_shards(handle) * 32
    return torch.as_tensor(DevicePtrView(sbf_filter_device_ptr(handle), n), device="cuda")


def or_allreduce_filter(handle, group=None, stream=None, window_bytes: int = 1 << 28) -> int:
    """The insert path's exchange step on GPUs: all-gather windows of the replicas over NCCL/NVLink,
    OR them in with the library's kernel."""
    from . import sbf_or_range_device

    def or_into(offset: int, chunk):
        sbf_or_range_device(handle, offset, chunk, chunk.numel(), stream)

    return or_allreduce(filter_tensor(handle), or_into, group=group, window_bytes=window_bytes)

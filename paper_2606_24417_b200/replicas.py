"""Multi-GPU plumbing for the replica scheme.

The path shards by input: every rank owns a private filter replica and a contiguous slice of the
insert batch (k-mer start positions, or whole records); after the local inserts ONE exchange step
makes the replicas identical — a bitwise-OR all-reduce of the filter bytes.  NCCL has no OR
reduction, so it is a reduce-scatter built from point-to-point exchanges plus the library's
``sbf_or_range_device`` kernel, followed by an in-place all-gather.  Queries then shard by reads with no collective at all.

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


def _slices(n: int, world: int):
    """Cut [0, n) (n a multiple of 32) in `world` contiguous slices on 32-byte (shard) boundaries."""
    shards = n // 32
    cuts = [32 * ((shards * r) // world) for r in range(world + 1)]
    return [(cuts[r], cuts[r + 1]) for r in range(world)]


def or_allreduce(local, or_into: Callable[[int, object], None], group=None, window_bytes: int = 1 << 28) -> int:
    """Make every rank's replica the OR of all replicas — a reduce-scatter followed by an all-gather, so that
    each rank sends and receives 2 (N-1)/N of the filter instead of the N-1 filters of a plain all-gather.

    local    : 1-D uint8 torch tensor viewing this rank's replica (device tensor under NCCL, CPU tensor under
               gloo), a multiple of 32 bytes long; updated in place.
    or_into  : callable(offset_bytes, peer_chunk_tensor) that ORs a peer's chunk into the local replica at that
               byte offset (sbf_or_range_device for the GPU path).
    Per window of the filter (scratch stays at window_bytes): (1) every rank sends slice j of its window to rank j
    (batched point-to-point) and ORs the N-1 slices it receives into its own slice; (2) the now final slices are
    all-gathered straight into the local replica (no kernel: the gather's outputs ARE views of the filter).
    Returns the number of OR calls issued.
    """
    import torch
    import torch.distributed as dist

    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    if world == 1:
        return 0
    n = local.numel()
    assert n % 32 == 0, "the filter is a whole number of 32-byte shards"
    window = min(n, max(32 * world, window_bytes - window_bytes % 32))
    scratch = torch.empty(window, dtype=torch.uint8, device=local.device)
    calls = 0
    for a in range(0, n, window):
        w = min(window, n - a)
        sl = _slices(w, world)
        my0, my1 = sl[rank]
        # (1) reduce-scatter: my slice of every peer's window arrives in scratch, one peer after the other
        ops, views, pos = [], [], 0
        for peer in range(world):
            if peer == rank:
                continue
            p0, p1 = sl[peer]
            if p1 > p0:
                ops.append(dist.P2POp(dist.isend, local[a + p0:a + p1], _global_rank(group, peer), group))
            if my1 > my0:
                v = scratch[pos:pos + (my1 - my0)]
                pos += my1 - my0
                views.append(v)
                ops.append(dist.P2POp(dist.irecv, v, _global_rank(group, peer), group))
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()
        for v in views:
            or_into(a + my0, v)
            calls += 1
        # (2) all-gather of the reduced slices, in place (slices may differ in length by one shard: gather by broadcast
        #     when they do, by one all_gather when they are equal)
        lens = {p1 - p0 for p0, p1 in sl}
        if len(lens) == 1 and my1 > my0:
            # in place: this rank's input IS slot `rank` of the output (the layout NCCL's in-place all-gather wants)
            dist.all_gather_into_tensor(local[a:a + w], local[a + my0:a + my1], group=group)
        else:
            for src in range(world):
                p0, p1 = sl[src]
                if p1 > p0:
                    dist.broadcast(local[a + p0:a + p1], _global_rank(group, src), group=group)
    return calls


def _global_rank(group, group_rank: int) -> int:
    import torch.distributed as dist
    return group_rank if group is None else dist.get_global_rank(group, group_rank)


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
    """The insert path's exchange step on GPUs: per window of the filter a reduce-scatter (batched NCCL
    point-to-point over NVLink + the library's OR kernel) and an in-place all-gather (see or_allreduce).

    Ordering: NCCL collectives synchronise with torch's CURRENT stream only, so the whole exchange runs with
    `stream` (the stream the inserts were enqueued on; None = the current one) made current: the sends then wait
    for the inserts, every OR kernel waits for its receive, and the next window's receives wait for the ORs that
    still read the scratch buffer."""
    import torch
    from . import sbf_or_range_device

    if stream is None:
        st = torch.cuda.current_stream()
    elif isinstance(stream, int):
        st = torch.cuda.ExternalStream(stream)
    else:
        st = stream

    def or_into(offset: int, chunk):
        sbf_or_range_device(handle, offset, chunk, chunk.numel(), st)

    with torch.cuda.stream(st):
        return or_allreduce(filter_tensor(handle), or_into, group=group, window_bytes=window_bytes)


# ---- peer-memory form of the exchange: each rank ORs its slice straight out of its peers' filters ---------------
def merge_plan(n_bytes: int, world: int, window_bytes: int = 1 << 28):
    """The windows and per-rank slices the exchange walks: [(window_offset, [(slice_lo, slice_hi) per rank])], all in
    bytes, slices relative to the window and cut on shard (32-byte) boundaries.  Pure arithmetic (tested on CPU)."""
    assert n_bytes % 32 == 0
    window = min(n_bytes, max(32 * world, window_bytes - window_bytes % 32))
    return [(a, _slices(min(window, n_bytes - a), world)) for a in range(0, n_bytes, window)]


def merge_local_replicas(handles, window_bytes: int = 1 << 28, stream=None) -> int:
    """Replicas that live on ONE device (e.g. filled on different streams): afterwards every one holds the OR of all.
    Walks the same plan as the multi-GPU exchange with the same kernels — `sbf_or_peers_range_device` reads the
    other replicas in place for the reduce-scatter step, the reduced slices are then copied back out — so a single
    GPU exercises the window / slice arithmetic and the peer-read kernel of `or_allreduce_filter_peer`.
    Returns the number of peer-read kernel launches."""
    import torch
    from . import sbf_filter_device_ptr, sbf_num_shards, sbf_or_peers_range_device

    world = len(handles)
    n = sbf_num_shards(handles[0]) * 32
    assert all(sbf_num_shards(h) * 32 == n for h in handles)
    base = [sbf_filter_device_ptr(h) for h in handles]
    tens = [filter_tensor(h) for h in handles]
    launches = 0
    ctx = torch.cuda.stream(stream) if stream is not None else _null_ctx()
    with ctx:
        for a, slices in merge_plan(n, world, window_bytes):
            for j, (lo, hi) in enumerate(slices):          # "rank" j reduces its slice of this window
                if hi > lo:
                    peers = [base[p] + a + lo for p in range(world) if p != j]
                    sbf_or_peers_range_device(handles[j], a + lo, peers, hi - lo, stream)
                    launches += 1
            for j, (lo, hi) in enumerate(slices):          # all-gather: every replica takes slice j from its owner
                for p in range(world):
                    if p != j and hi > lo:
                        tens[p][a + lo:a + hi].copy_(tens[j][a + lo:a + hi], non_blocking=True)
    return launches


class _null_ctx:
    def __enter__(self): return self
    def __exit__(self, *a): return False


def or_allreduce_filter_peer(handle, group=None, stream=None, window_bytes: int = 1 << 28) -> int:
    """The exchange over NVLink peer memory ("a peer-read reduce-scatter/all-gather kernel"): every
    rank maps its peers' filters through CUDA IPC once, then per window (1) ORs its own slice straight out of the
    peers' filters with ONE kernel (`sbf_or_peers_range_device`: N-1 remote reads per word, no receive buffer, no
    separate OR pass), (2) after a barrier copies the other ranks' finished slices out of their filters.  2 (N-1)/N
    filters cross NVLink per rank, as in the NCCL form, but without staging and with the reduce fused into the transfer.
    Ranks must share a node (CUDA IPC).  NEVER RUN ON MORE THAN ONE GPU in this repository's environment (one GPU per
    box): the plan and the kernel are exercised by `merge_local_replicas` on one device, the IPC mapping is not."""
    import torch
    import torch.distributed as dist
    from . import (sbf_filter_device_ptr, sbf_ipc_close_filter, sbf_ipc_export_filter, sbf_ipc_open_filter, sbf_num_shards,
                   sbf_or_peers_range_device)

    world, rank = dist.get_world_size(group), dist.get_rank(group)
    if world == 1:
        return 0
    st = torch.cuda.current_stream() if stream is None else (torch.cuda.ExternalStream(stream) if isinstance(stream, int) else stream)
    n = sbf_num_shards(handle) * 32
    mine = sbf_ipc_export_filter(handle)
    handles = [None] * world
    dist.all_gather_object(handles, mine, group=group)
    peer_ptr = {p: sbf_ipc_open_filter(handles[p]) for p in range(world) if p != rank}
    local = filter_tensor(handle)
    launches = 0
    try:
        with torch.cuda.stream(st):
            for a, slices in merge_plan(n, world, window_bytes):
                st.synchronize()
                dist.barrier(group=group)                       # every rank's inserts (or previous window) are done
                lo, hi = slices[rank]
                if hi > lo:
                    sbf_or_peers_range_device(handle, a + lo, [peer_ptr[p] + a + lo for p in peer_ptr], hi - lo, st)
                    launches += 1
                st.synchronize()
                dist.barrier(group=group)                       # all slices reduced: gather them
                for p, (plo, phi) in enumerate(slices):
                    if p != rank and phi > plo:
                        src = torch.as_tensor(DevicePtrView(peer_ptr[p] + a + plo, phi - plo), device="cuda")
                        local[a + plo:a + phi].copy_(src, non_blocking=True)
            st.synchronize()
            dist.barrier(group=group)                           # nobody unmaps while a peer still reads
    finally:
        for p in peer_ptr.values():
            sbf_ipc_close_filter(p)
    return launches

"""Multi-rank (world_size 2, gloo, CPU) test of the replica scheme's host logic:
partition of the insert batch + bitwise-OR all-reduce of the replicas == single-rank filter.
The per-rank filters come from the oracle (no GPU here); the product's kernels take the same
partitions and the same or_allreduce() on NCCL."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import seqgen
from paper_2606_24417_b200 import replicas

P = dict(k=31, m=16, s=28, H=4)
NUM_BITS = 1 << 20


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _workload():
    seq = seqgen.markov(31, 5, 0.41, 120_000)
    seq[40_000:40_200] = ord("N")
    offs = seqgen.record_offsets(7, seq.size, 9, 5_000, 30_000)
    return seq, offs


def _rank_main(rank, world, port, mode, out_dir, window=40_000):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        seq, offs = _workload()
        o = oracle.OracleSBF(num_bits=NUM_BITS, **P)
        if mode == "positions":
            a, e = replicas.partition_positions(seq.size, P["k"], world, rank)
            if e > a:
                o.insert_records(seq[a:e])
        else:
            r0, r1 = replicas.partition_records(offs, world, rank)
            if r1 > r0:
                o.insert_records(seq[int(offs[r0]):int(offs[r1])], replicas.rebase_offsets(offs, r0, r1))
        words = o.words().reshape(-1)
        local = torch.from_numpy(words.view(np.uint8))

        def or_into(offset, chunk):
            c = chunk.numpy()
            dst = words.view(np.uint8)[offset:offset + c.size]
            np.bitwise_or(dst, c, out=dst)

        calls = replicas.or_allreduce(local, or_into, window_bytes=window)  # several windows, last one ragged
        assert calls == (world - 1) * -(-local.numel() // (window - window % 32))  # one OR per peer per window
        np.save(os.path.join(out_dir, "rank%d.npy" % rank), o.export_bits())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("mode,world,window", [("positions", 2, 40_000), ("records", 2, 65_536), ("positions", 3, 40_000),
                                               ("records", 4, 16_384)])
def test_partition_plus_or_allreduce_equals_single_rank(tmp_path, mode, world, window):
    mp.spawn(_rank_main, args=(world, _free_port(), mode, str(tmp_path), window), nprocs=world, join=True)
    seq, offs = _workload()
    ref = oracle.OracleSBF(num_bits=NUM_BITS, **P)
    if mode == "positions":
        ref.insert_records(seq)
    else:
        ref.insert_records(seq, offs)
    want = ref.export_bits()
    for r in range(world):
        got = np.load(os.path.join(str(tmp_path), "rank%d.npy" % r))
        assert np.array_equal(got, want), "rank %d replica differs from the single-rank filter" % r


@pytest.mark.parametrize("total,k,world", [(0, 31, 4), (10, 31, 4), (31, 31, 3), (1000, 31, 1), (1000, 31, 7), (12345, 9, 8)])
def test_partition_positions_covers_every_kmer_start_once(total, k, world):
    starts = np.zeros(max(total - k + 1, 0), dtype=np.int32)
    for r in range(world):
        a, e = replicas.partition_positions(total, k, world, r)
        assert 0 <= a <= e <= total
        if e - a >= k:
            starts[a:e - k + 1] += 1   # k-mer starts complete inside [a, e)
    assert (starts == 1).all()


@pytest.mark.parametrize("world", [1, 2, 3, 8, 40])
def test_partition_records_is_a_partition(world):
    offs = seqgen.record_offsets(5, 1_000_000, 24, 10_000, 90_000)
    cuts = [replicas.partition_records(offs, world, r) for r in range(world)]
    assert cuts[0][0] == 0 and cuts[-1][1] == 24
    for (a0, a1), (b0, b1) in zip(cuts, cuts[1:]):
        assert a1 == b0 and a0 <= a1
    sizes = [int(offs[b]) - int(offs[a]) for a, b in cuts]
    if world <= 8:
        assert max(sizes) <= 1_000_000 / world + 90_000
    reb = replicas.rebase_offsets(offs, *cuts[0])
    assert reb[0] == 0 and reb[-1] == sizes[0]

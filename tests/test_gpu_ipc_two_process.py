"""The peer-memory replica merge (replicas.or_allreduce_filter_peer) executed across PROCESSES.

One GPU per box is all this repository's environment has, so the merge has never crossed NVLink; what CAN run for real
is everything else: two (or three) processes, each with a filter of its own on the one GPU, exchange
sbf_ipc_export_filter handles through a gloo process group, map each other's filters with sbf_ipc_open_filter, reduce
their slice of every window straight out of the peers' mapped memory with sbf_or_peers_range_device, gather the reduced
slices through the same mappings, and unmap.  The ranks only ever wait for each other on the HOST (gloo barriers between
stream-synchronised phases); no kernel waits for another process's kernel.

Expected values come from the oracle alone: every rank's merged replica must equal the oracle's filter after inserting
the whole batch, and a query on any rank must give the oracle's bitmap."""
import os
import socket

import numpy as np
import pytest

import oracle
import seqgen

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

P = dict(k=31, m=16, s=28, H=4)
NUM_BITS = 1 << 23          # 1 MiB of filter: several windows of 192 KiB, the last one ragged


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _workload():
    seq = seqgen.markov(31, 5, 0.41, 600_000)
    seq[150_000:150_400] = ord("N")
    offs = seqgen.record_offsets(7, seq.size, 11, 20_000, 120_000)
    return seq, offs


def _rank_main(rank, world, port, mode, window, out_dir):
    import torch.distributed as dist
    import paper_2606_24417_b200 as sbf
    from paper_2606_24417_b200 import replicas
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        torch.cuda.set_device(0)                       # every rank on the one GPU
        seq, offs = _workload()
        with sbf.SuperBloomFilter(num_bits=NUM_BITS, **P) as f:
            st = torch.cuda.Stream()
            if mode == "positions":
                a, e = replicas.partition_positions(seq.size, P["k"], world, rank)
                d = torch.from_numpy(seq[a:e].copy()).cuda()
                sbf.sbf_insert_seq(f.handle, d, d.numel(), st)
            else:
                r0, r1 = replicas.partition_records(offs, world, rank)
                d = torch.from_numpy(seq[int(offs[r0]):int(offs[r1])].copy()).cuda()
                o = torch.from_numpy(replicas.rebase_offsets(offs, r0, r1).view(np.int64)).cuda()
                sbf.sbf_insert_records(f.handle, d, o, r1 - r0, d.numel(), st)
            before = f.export_bits()                   # this rank's share only (synchronises)
            launches = replicas.or_allreduce_filter_peer(f.handle, stream=st, window_bytes=window)
            st.synchronize()
            n_windows = -(-(NUM_BITS // 8) // (window - window % 32))
            assert launches == n_windows, (launches, n_windows)
            np.save(os.path.join(out_dir, "before%d.npy" % rank), before)
            np.save(os.path.join(out_dir, "rank%d.npy" % rank), f.export_bits())
            # the merged replica answers queries for k-mers another rank inserted
            bm = torch.full(((seq.size + 31) // 32,), -1, dtype=torch.int32, device="cuda")
            dq = torch.from_numpy(seq).cuda()
            sbf.sbf_query_seq(f.handle, dq, dq.numel(), bm)
            torch.cuda.synchronize()
            np.save(os.path.join(out_dir, "bitmap%d.npy" % rank), bm.cpu().numpy().view(np.uint32))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("mode,world,window", [("positions", 2, 196_608), ("records", 2, 1 << 28), ("positions", 3, 100_000)])
def test_peer_memory_merge_across_processes(tmp_path, mode, world, window):
    import torch.multiprocessing as mp
    mp.spawn(_rank_main, args=(world, _free_port(), mode, window, str(tmp_path)), nprocs=world, join=True)
    seq, offs = _workload()
    ref = oracle.OracleSBF(num_bits=NUM_BITS, **P)
    ref.insert_records(seq, None if mode == "positions" else offs, threads=True)
    want = ref.export_bits()
    wbm, _, _ = ref.query_records(seq, None, threads=True)      # the whole sequence as one record, on every rank
    union = np.zeros_like(want)
    for r in range(world):
        before = np.load(os.path.join(str(tmp_path), "before%d.npy" % r))
        assert before.any() and not np.array_equal(before, want), "rank %d's share is not a proper part" % r
        union |= before
        got = np.load(os.path.join(str(tmp_path), "rank%d.npy" % r))
        assert np.array_equal(got, want), "rank %d: merged replica differs from the oracle's single filter in %d bytes" % (
            r, np.count_nonzero(got != want))
        assert np.array_equal(np.load(os.path.join(str(tmp_path), "bitmap%d.npy" % r)), wbm), "rank %d: query bitmap" % r
    assert np.array_equal(union, want)
    ref.close()

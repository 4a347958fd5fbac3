"""Record-mode query batches that hold records too long for one thread (above 1024 symbols).

stream_rec_kernel lists such records, stream_long_kernel walks only them, chunk by chunk; the short records' results
stand ("dense record batch": no k-mer spans two records).  Until round 3 one long record made the chunk
kernels redo the whole batch.  Bitmap words and per-record counts are compared with the oracle, tolerance 0; the
timing case shows that the cost follows the long records' symbols, not the batch."""
import json
import os

import numpy as np
import pytest

import oracle
import seqgen
import paper_2606_24417_b200 as sbf

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

DEFAULT = dict(k=31, m=16, s=28, H=4)
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _batch(genome, lens, seed):
    """Records of the given lengths: even ones cut from the genome at seeded places (hits), odd ones uniform."""
    rng = np.random.default_rng(seed)
    offs = np.concatenate(([0], np.cumsum(lens))).astype(np.uint64)
    out = seqgen.uniform(seed, int(offs[-1]))
    for i in range(0, len(lens), 2):
        L = int(lens[i])
        if 0 < L <= genome.size:
            s = int(rng.integers(0, genome.size - L + 1))
            out[int(offs[i]):int(offs[i]) + L] = genome[s:s + L]
    return out, offs


def _check(params, num_bits, genome, q, offs, expect_launches=None):
    o = oracle.OracleSBF(num_bits=num_bits, **params)
    o.insert_records(genome, threads=True)
    wbm, wc, _ = o.query_records(q, offs, threads=True)
    o.close()
    n_rec = offs.size - 1
    with sbf.SuperBloomFilter(num_bits=num_bits, **params) as f:
        assert f.specialized
        d = _dev(genome)
        sbf.sbf_insert_seq(f.handle, d, d.numel())
        dq, do = _dev(q), _dev(offs.view(np.int64))
        for rep in range(2):                                        # twice: the list and its counter are reused
            bm = torch.full(((q.size + 31) // 32,), -1, dtype=torch.int32, device="cuda")
            hc = torch.full((n_rec,), -1, dtype=torch.int32, device="cuda")
            n0 = sbf.sbf_kernel_launches()
            sbf.sbf_query_records(f.handle, dq, do, n_rec, q.size, bm, hc)
            torch.cuda.synchronize()
            if expect_launches is not None:
                assert sbf.sbf_kernel_launches() - n0 == expect_launches
            got = bm.cpu().numpy().view(np.uint32)
            if not np.array_equal(got, wbm):
                bad = np.flatnonzero(got != wbm)
                raise AssertionError("bitmap differs in %d words, first %d (record %d): got %08x want %08x" % (
                    bad.size, bad[0], int(np.searchsorted(offs, bad[0] * 32, side="right")) - 1, got[bad[0]], wbm[bad[0]]))
            gc = hc.cpu().numpy().view(np.uint32)
            if not np.array_equal(gc, wc):
                bad = np.flatnonzero(gc != wc)
                raise AssertionError("counts differ for %d records, first %d (length %d): got %d want %d" % (
                    bad.size, bad[0], int(offs[bad[0] + 1] - offs[bad[0]]), gc[bad[0]], wc[bad[0]]))
    return wc


@pytest.mark.parametrize("params", [DEFAULT, dict(k=31, m=12, s=24, H=8), dict(k=63, m=31, s=60, H=4)])
def test_long_records_among_short_reads(params):
    """Long records first, last, adjacent to each other, just above the limit, spanning many chunk groups, with N runs
    and with ends on and off the 128-position grid."""
    genome = seqgen.markov(31, 5, 0.41, 900_000)
    genome[400_000:400_300] = ord("N")
    lens = np.full(30_000, 150, dtype=np.int64)
    lens[0] = 1025                      # first record, just above the limit
    lens[1] = 1024                      # at the limit: still one thread
    lens[100] = 5000
    lens[101] = 16_384 + 7              # more than one group of 128 chunks... (128 * 128 = 16384 positions)
    lens[102] = 2000                    # three long records in a row
    lens[103] = 0
    lens[5000] = 300_000                # 19 groups; cut from the genome with its N run when even-indexed
    lens[9999] = 1100
    lens[29_999] = 70_001               # last record
    lens[20_000:20_050] = 64            # short ones around k
    q, offs = _batch(genome, lens, 77)
    assert (offs[-1] / (offs.size - 1)) <= 400      # record mode is tried (mean length)
    wc = _check(params, 1 << 24, genome, q, offs, expect_launches=6)  # pack, rec, long + the three idle fallback launches
    assert wc[5000] > 200_000 and wc[100] > 4000    # the long genome cuts are found


def test_long_record_list_overflow_falls_back_to_the_chunk_kernels():
    """More long records than the list holds (65536 groups): the flag goes up and the chunk kernels redo the batch,
    striding over it with their capped grid."""
    genome = seqgen.markov(32, 5, 0.41, 500_000)
    n_long, n_short = 66_000, 120_000
    lens = np.concatenate((np.full(n_long, 1025, dtype=np.int64), np.full(n_short, 40, dtype=np.int64)))
    np.random.default_rng(5).shuffle(lens)
    q, offs = _batch(genome, lens, 78)
    assert (offs[-1] / (offs.size - 1)) <= 400
    _check(DEFAULT, 1 << 24, genome, q, offs)


def test_cost_follows_the_long_records_not_the_batch():
    """1e6 reads of 150 plus 0, 1, 100 and 10 000 records of 5000 symbols: device time per query.  One long record must
    not cost a second pass over the batch (it did: 2x); 10 000 of them add 50 Mbp of work to 150 Mbp."""
    w = seqgen.config3(scale=0.1)
    n_reads = 1_000_000
    reads = w.read_batch(0, n_reads)
    times = {}
    with sbf.SuperBloomFilter(num_bits=1 << 30, **DEFAULT) as f:
        d = _dev(w.insert_bases)
        sbf.sbf_insert_seq(f.handle, d, d.numel())
        for n_long in (0, 1, 100, 10_000):
            lens = np.concatenate((np.full(n_reads, 150, dtype=np.int64), np.full(n_long, 5000, dtype=np.int64)))
            offs = np.concatenate(([0], np.cumsum(lens))).astype(np.uint64)
            q = np.concatenate((reads, seqgen.uniform(9, 5000 * n_long)))
            dq, do = _dev(q), _dev(offs.view(np.int64))
            bm = torch.empty((q.size + 31) // 32, dtype=torch.int32, device="cuda")
            hc = torch.empty(offs.size - 1, dtype=torch.int32, device="cuda")
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            best = 1e9
            for rep in range(6):
                ev[0].record()
                sbf.sbf_query_records(f.handle, dq, do, offs.size - 1, q.size, bm, hc)
                ev[1].record()
                torch.cuda.synchronize()
                if rep:
                    best = min(best, ev[0].elapsed_time(ev[1]))
            times[n_long] = best
    out = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(out):
        with open(os.path.join(out, "long_records_timing.json"), "w") as fh:
            json.dump(times, fh)
    assert times[1] < 1.10 * times[0], times
    assert times[100] < 1.15 * times[0], times
    assert times[10_000] < 1.8 * times[0], times       # +33 % symbols, walked at the chunk kernels' rate

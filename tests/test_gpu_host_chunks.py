"""GPU parity of the HOST-facing calls when a batch is cut in several staged chunks (the path bench.py's `e2e` times).

`sbf_set_host_chunk` shrinks the chunk so that a small batch exercises everything the 32 Mi default does at full
size: the k-1 overlap, records that straddle a chunk edge (boundaries before, on and inside the overlap), a record
longer than a chunk, empty records on an edge, the two alternating staging slots and their event waits (>= 3
chunks), the per-chunk offsets rebased on the device, the bitmap word shared by two chunks and the per-chunk D2H
window.  One test runs the default 32 Mi chunks on >= 70 Mi symbols.  Everything is compared with the oracle, bit for
bit, on poisoned output buffers, from pageable and from pinned caller memory."""
import numpy as np
import pytest

import oracle
import seqgen
import paper_2606_24417_b200 as sbf

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

DEFAULT = dict(k=31, m=16, s=28, H=4)


def _pin(a):
    t = torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    return t, t.numpy()


def _edge_offsets(total, chunk, k, rng):
    """Record boundaries placed around every chunk edge: just before it, on it, inside the k-1 overlap, just after
    the overlap; plus ragged short records, empty records on an edge, and one record longer than a chunk."""
    cuts = set()
    n_chunks = total // chunk
    deltas = [-1, 0, 1, 15, k - 2, k - 1, k, k + 1, 40]
    for c in range(1, n_chunks + 1):
        d = deltas[c % len(deltas)]
        if 0 < c * chunk + d < total:
            cuts.add(c * chunk + d)
    lo = 2 * chunk + 100                                    # a record longer than a chunk: nothing cut in here
    hi = lo + chunk + 700
    pos = 0
    while pos < total:
        pos += int(rng.integers(1, 400))
        if pos < total and not (lo < pos < hi):
            cuts.add(pos)
    cuts = sorted(c for c in cuts if not (lo < c < hi))
    offs = [0]
    for c in cuts:
        offs.append(c)
        if c % chunk == 0 or rng.random() < 0.03:
            offs.extend([c, c])                             # empty records, some exactly on a chunk edge
    offs.append(total)
    return np.array(offs, dtype=np.uint64)


def _check_host_paths(params, num_bits, chunk, ins, ins_offs, q, q_offs, pinned):
    o = oracle.OracleSBF(num_bits=num_bits, **params)
    o_rec = oracle.OracleSBF(num_bits=num_bits, **params)
    o.insert_records(ins, threads=True)
    o_rec.insert_records(ins, ins_offs, threads=True)
    want_bm, want_counts, _ = o.query_records(q, q_offs, threads=True)
    want_bm_seq, want_c_seq, _ = o.query_records(q, None, threads=True)
    keep = []
    if pinned:
        t, ins_h = _pin(ins); keep.append(t)
        t, q_h = _pin(q); keep.append(t)
        t, qo_h = _pin(q_offs.view(np.int64)); keep.append(t)
        qo_h = qo_h.view(np.uint64)
        t, io_h = _pin(ins_offs.view(np.int64)); keep.append(t)
        io_h = io_h.view(np.uint64)
    else:
        ins_h, q_h, qo_h, io_h = ins, q, q_offs, ins_offs
    with sbf.SuperBloomFilter(num_bits=num_bits, **params) as f:
        if chunk:
            sbf.sbf_set_host_chunk(f.handle, chunk)
        # insert as records
        sbf.sbf_insert_records_host(f.handle, ins_h, io_h, io_h.size - 1)
        got = f.export_bits()
        assert np.array_equal(got, o_rec.export_bits()), "sbf_insert_records_host: filter differs from the oracle"
        # insert as one sequence
        f.clear()
        sbf.sbf_insert_seq_host(f.handle, ins_h, ins_h.size)
        assert np.array_equal(f.export_bits(), o.export_bits()), "sbf_insert_seq_host: filter differs from the oracle"
        # query as records (poisoned outputs)
        bm = np.full((q.size + 31) // 32, 0xFFFFFFFF, dtype=np.uint32)
        hc = np.full(q_offs.size - 1, 0xFFFFFFFF, dtype=np.uint32)
        sbf.sbf_query_records_host(f.handle, q_h, qo_h, qo_h.size - 1, bm, hc)
        bad = np.flatnonzero(bm != want_bm)
        assert bad.size == 0, "sbf_query_records_host: %d bitmap words differ, first %d (symbol %d)" % (
            bad.size, bad[0], 32 * bad[0])
        assert np.array_equal(hc, want_counts), "sbf_query_records_host: hit counts differ"
        # query as one sequence
        bm2 = np.full_like(bm, 0xFFFFFFFF)
        hits = np.full(1, 0xFFFFFFFFFFFFFFFF, dtype=np.uint64)
        sbf.sbf_query_seq_host(f.handle, q_h, q_h.size, bm2, hits)
        assert np.array_equal(bm2, want_bm_seq), "sbf_query_seq_host: bitmap differs"
        assert int(hits[0]) == int(want_c_seq.sum())
    o.close(); o_rec.close()


@pytest.mark.parametrize("pinned", [False, True])
@pytest.mark.parametrize("chunk", [4096, 1152])
def test_small_chunks_all_edge_placements(chunk, pinned):
    rng = np.random.default_rng(chunk + int(pinned))
    total = 13 * chunk + 777                       # 14 chunks, the last one ragged
    ins = seqgen.markov(31, 5, 0.41, total)
    ins[3 * chunk - 5:3 * chunk + 9] = ord("N")     # an N run across a chunk edge
    ins_offs = _edge_offsets(total, chunk, 31, rng)
    q = seqgen.uniform(77, total)
    q[: total // 2] = ins[: total // 2]             # true members in the first half (incl. the long record)
    q[5 * chunk + 3] = ord("N")
    q_offs = _edge_offsets(total, chunk, 31, rng)
    _check_host_paths(DEFAULT, 1 << 22, chunk, ins, ins_offs, q, q_offs, pinned)


@pytest.mark.parametrize("params", [dict(k=21, m=11, s=21, H=3), dict(k=31, m=12, s=24, H=8), dict(k=31, m=16, s=28, H=12)])
def test_small_chunks_other_parameters(params):
    """Other k (different overlap), the general-Z kernels and the runtime-parameter kernel behind the same staging."""
    chunk = 2048
    rng = np.random.default_rng(5)
    total = 7 * chunk + 31
    ins = seqgen.uniform(3, total)
    q = seqgen.uniform(4, total); q[1000:9000] = ins[1000:9000]
    _check_host_paths(params, 1 << 20, chunk, ins, _edge_offsets(total, chunk, params["k"], rng), q,
                      _edge_offsets(total, chunk, params["k"], rng), False)


def test_more_empty_records_than_symbols():
    """Empty records repeat an offset: a chunk can hold more record boundaries than symbols (the per-chunk offsets
    buffer is sized by records, not by symbols)."""
    rng = np.random.default_rng(9)
    lens = np.zeros(5000, dtype=np.int64)
    lens[rng.choice(5000, 12, replace=False)] = rng.integers(31, 200, 12)
    offs = np.concatenate(([0], np.cumsum(lens))).astype(np.uint64)
    total = int(offs[-1])
    bases = seqgen.uniform(8, total)
    o = oracle.OracleSBF(num_bits=1 << 18, **DEFAULT)
    o.insert_records(bases, offs)
    want_bm, want_c, _ = o.query_records(bases, offs)
    for chunk in (0, 256):
        with sbf.SuperBloomFilter(num_bits=1 << 18, **DEFAULT) as f:
            if chunk:
                sbf.sbf_set_host_chunk(f.handle, chunk)
            sbf.sbf_insert_records_host(f.handle, bases, offs, offs.size - 1)
            assert np.array_equal(f.export_bits(), o.export_bits())
            bm = np.full((total + 31) // 32, 0xFFFFFFFF, dtype=np.uint32)
            hc = np.full(offs.size - 1, 0xFFFFFFFF, dtype=np.uint32)
            sbf.sbf_query_records_host(f.handle, bases, offs, offs.size - 1, bm, hc)
            assert np.array_equal(bm, want_bm) and np.array_equal(hc, want_c)
            assert int(hc.sum()) == int(want_c.sum()) > 0
    o.close()


@pytest.mark.slow
def test_default_32mi_chunks_three_chunks():
    """The default chunk size on > 70 Mi symbols (3 chunks): 150-base reads straddle both 32 Mi edges (150 does not
    divide 2^25) and one record is longer than a chunk, so the device-side fallback behind record mode runs too."""
    chunk = 32 << 20
    n_a, long_len, n_b = 120_000, chunk + 1_000_003, 150_000
    w = seqgen.config3(scale=0.3)                          # 75 Mbp with N runs
    ins = w.insert_bases
    assert ins.size > 2 * chunk
    lens = np.concatenate((np.full(n_a, 150), [long_len], np.full(n_b, 150))).astype(np.int64)
    q_offs = np.concatenate(([0], np.cumsum(lens))).astype(np.uint64)
    total = int(q_offs[-1])
    assert total > 70 << 20 and total // chunk == 2
    q = np.empty(total, dtype=np.uint8)
    q[: n_a * 150] = w.read_batch(0, n_a)
    a = n_a * 150
    q[a:a + long_len] = ins[5_000_000:5_000_000 + long_len]          # the long record: all true members
    q[a + long_len:] = w.read_batch(n_a, n_b)
    nb = 1 << 30
    o = oracle.OracleSBF(num_bits=nb, **DEFAULT)
    o.insert_records(ins, threads=True)
    want_bm, want_c, _ = o.query_records(q, q_offs, threads=True)
    t_ins, ins_h = _pin(ins)
    t_q, q_h = _pin(q)
    with sbf.SuperBloomFilter(num_bits=nb, **DEFAULT) as f:
        sbf.sbf_insert_seq_host(f.handle, ins_h, ins_h.size)
        got, want = f.export_bits(), o.export_bits()
        assert np.array_equal(got, want), "filter differs in %d bytes" % np.count_nonzero(got != want)
        bm = np.full((total + 31) // 32, 0xFFFFFFFF, dtype=np.uint32)
        hc = np.full(q_offs.size - 1, 0xFFFFFFFF, dtype=np.uint32)
        sbf.sbf_query_records_host(f.handle, q_h, q_offs, q_offs.size - 1, bm, hc)
        bad = np.flatnonzero(bm != want_bm)
        assert bad.size == 0, "%d bitmap words differ, first at symbol %d" % (bad.size, 32 * bad[0])
        assert np.array_equal(hc, want_c)
        assert int(hc[n_a]) > 0.95 * (long_len - 30)       # the long record is a copy of inserted sequence (minus N runs)
    o.close()

"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(one sbf_insert_seq over the whole sequence, one sbf_query_records per 4e6-read batch, 2^32-bit filter).
The oracle's OpenMP driver (pinned equal to the single-threaded definition by P6) makes the full
comparison affordable: every filter byte, every bitmap word and every hit count, tolerance 0."""
import numpy as np
import pytest

import oracle
import seqgen
import paper_2606_24417_b200 as sbf

torch = pytest.importorskip("torch")
pytestmark = [pytest.mark.gpu, pytest.mark.slow]

DEFAULT = dict(k=31, m=16, s=28, H=4)


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _first_diff(got, want, what):
    if np.array_equal(got, want):
        return
    bad = np.flatnonzero(got != want)
    raise AssertionError("%s differs in %d of %d elements, first at %d: got %r want %r" %
                         (what, bad.size, got.size, bad[0], got[bad[0]], want[bad[0]]))


def _query_every_batch(f, o, w, batch, max_fpr):
    """All of the workload's reads, batch by batch (bench.py's launch: one sbf_query_records per `batch` reads, device
    buffers reused): every bitmap word and every per-read count of every batch against the oracle's OpenMP driver.
    Per batch also the property that holds at any size: the error-free k-mers of the sampled reads are
    all reported present, i.e. a sampled read's count is never below what its substitutions can explain."""
    k, L = DEFAULT["k"], w.read_len
    per = L - k + 1
    assert w.n_reads % batch == 0
    offs = seqgen.fixed_offsets(batch, L)
    d_offs = _dev(offs.view(np.int64))
    reads = np.empty(batch * L, dtype=np.uint8)
    d_reads = torch.empty(batch * L, dtype=torch.uint8, device="cuda")
    bm = torch.empty((batch * L + 31) // 32, dtype=torch.int32, device="cuda")
    hc = torch.empty(batch, dtype=torch.int32, device="cuda")
    n_batches = w.n_reads // batch
    for b in range(n_batches):
        w.read_batch(b * batch, batch, out=reads)
        d_reads.copy_(torch.from_numpy(reads))
        bm.fill_(-1)
        hc.fill_(-1)
        f.query_records(d_reads, d_offs, bm, hc)
        torch.cuda.synchronize()
        wbm, wc, _ = o.query_records(reads, offs, threads=True)
        _first_diff(bm.cpu().numpy().view(np.uint32), wbm, "batch %d of %d: bitmap words" % (b, n_batches))
        got_c = hc.cpu().numpy().view(np.uint32)
        _first_diff(got_c, wc, "batch %d of %d: hit counts" % (b, n_batches))
        # sampled reads (even index): mostly present; uniform reads (odd index): only false positives
        assert got_c[0::2].astype(np.int64).sum() > 0.6 * (batch // 2) * per, b
        assert got_c[1::2].astype(np.int64).sum() < max_fpr * (batch // 2) * per, b
        # a sampled read without any substitution that lies clear of N runs has all its k-mers present
        for r in range(0, 2000, 2):
            g = b * batch + r
            if any(seqgen.read_is_sub(w.read_seed, w.read_sub_rate, L, g, i) for i in range(L)):
                continue
            start = seqgen.read_start(w.read_seed, w.insert_bases.size, L, g)
            src = w.insert_bases[start:start + L]
            if np.isin(src, np.frombuffer(b"ACGT", dtype=np.uint8)).all() and _inside_one_record(w, start, L):
                assert got_c[r] == per, (b, r, int(got_c[r]))
    return n_batches


def _inside_one_record(w, start, length):
    o = w.insert_offsets
    r = int(np.searchsorted(o, start, side="right")) - 1
    return start + length <= int(o[r + 1])


_c3 = {}


def _config3():
    """The config-3 workload, generated once per session (250 Mbp, N runs)."""
    if "w" not in _c3:
        _c3["w"] = seqgen.config3()
    return _c3["w"]


def test_config3_full_size_filter_bitmap_counts():
    """BASELINE config 3 at full size: every filter byte after the 250 Mbp insert, then ALL 4e7 reads in bench.py's
    batches of 4e6 (10 batches): every bitmap word and every per-read count."""
    w = _config3()                             # 250 Mbp, N runs, 2^32-bit filter
    nb = w.params["num_bits"]
    assert w.n_reads == 40_000_000
    o = oracle.OracleSBF(num_bits=nb, **DEFAULT)
    n_ins = o.insert_records(w.insert_bases, threads=True)
    assert 240_000_000 < n_ins < 250_000_000
    with sbf.SuperBloomFilter(num_bits=nb, **DEFAULT) as f:
        assert f.specialized and f.num_shards == o.num_shards == 1 << 24
        d_seq = _dev(w.insert_bases)
        f.insert_seq(d_seq)
        torch.cuda.synchronize()
        _first_diff(f.export_bits(), o.export_bits(), "filter bytes")
        del d_seq
        assert _query_every_batch(f, o, w, 4_000_000, max_fpr=1e-3) == 10     # 17 bits per inserted k-mer
    o.close()


def test_config4_shape_4gib_filter_multi_record():
    """2^35-bit filter (P = 27 shards, 64-bit byte offsets) with a 24-record insert at 1/25 scale."""
    w = seqgen.config4(scale=0.04, n_reads=200_000)   # 124 Mbp in 24 records
    nb = 1 << 35
    o = oracle.OracleSBF(num_bits=nb, **DEFAULT)
    o.insert_records(w.insert_bases, w.insert_offsets, threads=True)
    with sbf.SuperBloomFilter(num_bits=nb, **DEFAULT) as f:
        assert f.num_shards == 1 << 27
        f.insert_records(_dev(w.insert_bases), _dev(w.insert_offsets.view(np.int64)))
        torch.cuda.synchronize()
        _first_diff(f.export_bits(), o.export_bits(), "filter bytes")
        reads = w.read_batch(0, 200_000)
        offs = seqgen.fixed_offsets(200_000, w.read_len)
        bm = torch.full(((reads.size + 31) // 32,), -1, dtype=torch.int32, device="cuda")
        hc = torch.full((200_000,), -1, dtype=torch.int32, device="cuda")
        f.query_records(_dev(reads), _dev(offs.view(np.int64)), bm, hc)
        torch.cuda.synchronize()
        wbm, wc, _ = o.query_records(reads, offs, threads=True)
        _first_diff(bm.cpu().numpy().view(np.uint32), wbm, "bitmap words")
        _first_diff(hc.cpu().numpy().view(np.uint32), wc, "hit counts")
    o.close()


def test_config2_full_size():
    w = seqgen.config2()
    distinct = seqgen.count_distinct_windows(w.insert_bases, DEFAULT["k"])  # exact (plain string set)
    assert 4_500_000 < distinct < 5_000_000
    nb = 16 * distinct
    reads = w.read_batch(0, w.n_reads)
    offs = seqgen.fixed_offsets(w.n_reads, w.read_len)
    o = oracle.OracleSBF(num_bits=nb, **DEFAULT)
    o.insert_records(w.insert_bases, threads=True)
    with sbf.SuperBloomFilter(num_bits=nb, **DEFAULT) as f:
        assert f.num_shards == o.num_shards == 1 << 19
        f.insert_seq(_dev(w.insert_bases))
        torch.cuda.synchronize()
        _first_diff(f.export_bits(), o.export_bits(), "filter bytes")
        bm = torch.full(((reads.size + 31) // 32,), -1, dtype=torch.int32, device="cuda")
        hc = torch.full((w.n_reads,), -1, dtype=torch.int32, device="cuda")
        f.query_records(_dev(reads), _dev(offs.view(np.int64)), bm, hc)
        torch.cuda.synchronize()
        wbm, wc, _ = o.query_records(reads, offs, threads=True)
        _first_diff(bm.cpu().numpy().view(np.uint32), wbm, "bitmap words")
        _first_diff(hc.cpu().numpy().view(np.uint32), wc, "hit counts")
    o.close()


def test_timing_abi_reports_kernel_times():
    seq = seqgen.uniform(5, 2_000_000)
    with sbf.SuperBloomFilter(num_bits=1 << 26, **DEFAULT) as f:
        with pytest.raises(sbf.SBFError):
            sbf.sbf_get_timing(f.handle)          # timing is off
        sbf.sbf_set_timing(f.handle, True)
        with pytest.raises(sbf.SBFError):
            sbf.sbf_get_timing(f.handle)          # no timed call yet
        d = _dev(seq)
        f.insert_seq(d)
        pack_ms, main_ms, count_ms = sbf.sbf_get_timing(f.handle)
        assert pack_ms > 0 and main_ms > 0 and count_ms == 0
        bm = torch.empty((seq.size + 31) // 32, dtype=torch.int32, device="cuda")
        hits = torch.zeros(1, dtype=torch.int64, device="cuda")
        f.query_seq(d, bm, hits)
        pack_ms, main_ms, count_ms = sbf.sbf_get_timing(f.handle)
        assert pack_ms > 0 and main_ms > 0 and count_ms > 0
        assert int(hits.item()) == seq.size - DEFAULT["k"] + 1
        n0 = sbf.sbf_kernel_launches()
        f.insert_seq(d)
        assert sbf.sbf_kernel_launches() - n0 == 2   # pack + fused insert kernel


def test_config4_full_size_insert_and_query_batch():
    """BASELINE config 4 at full size: 3.1 Gbp in 24 records into a 2^35-bit filter (every one of the 4 GiB filter
    bytes compared), then ALL 1e8 reads in batches of 4e6 (25 batches): every bitmap word and every per-read count."""
    w = seqgen.config4()
    nb = w.params["num_bits"]
    assert w.n_reads == 100_000_000
    o = oracle.OracleSBF(num_bits=nb, **DEFAULT)
    n_ins = o.insert_records(w.insert_bases, w.insert_offsets, threads=True)
    assert n_ins > 3_000_000_000
    with sbf.SuperBloomFilter(num_bits=nb, **DEFAULT) as f:
        assert f.num_shards == o.num_shards == 1 << 27
        d_ins = _dev(w.insert_bases)
        f.insert_records(d_ins, _dev(w.insert_offsets.view(np.int64)))
        torch.cuda.synchronize()
        del d_ins
        got = f.export_bits()
        want = o.words().reshape(-1).view(np.uint8)
        step = 1 << 28
        for a in range(0, got.size, step):                  # compare in slices: no third 4 GiB copy
            _first_diff(got[a:a + step], want[a:a + step], "filter bytes [%d, +%d)" % (a, step))
        del got
        assert _query_every_batch(f, o, w, 4_000_000, max_fpr=2e-2) == 25     # 11 bits per inserted k-mer: FPR 0.7 %
    o.close()


def test_config3_chunk_mode_query_of_the_inserted_sequence():
    """sbf_query_seq of long sequences runs the CHUNK-mode query kernel; its chunk length depends on the batch size
    (chunk_blocks 8 from 64 Mi symbols, 4 from 16 Mi).  Config 1's "query the same sequence" at config-3 size: the
    whole 250 Mbp sequence against its own 2^32-bit filter (chunk_blocks 8) and a 20 Mbp stretch (chunk_blocks 4);
    bitmap equal to the oracle's and every valid k-mer true."""
    w = _config3()
    nb = w.params["num_bits"]
    o = oracle.OracleSBF(num_bits=nb, **DEFAULT)
    o.insert_records(w.insert_bases, threads=True)
    with sbf.SuperBloomFilter(num_bits=nb, **DEFAULT) as f:
        d_seq = _dev(w.insert_bases)
        f.insert_seq(d_seq)
        for a, n in ((0, w.insert_bases.size), (100_000_000, 20_000_000)):
            assert n >= (64 << 20) or (16 << 20) <= n < (64 << 20)
            view = d_seq[a:a + n]
            bm = torch.full(((n + 31) // 32,), -1, dtype=torch.int32, device="cuda")
            hits = torch.full((1,), -1, dtype=torch.int64, device="cuda")
            sbf.sbf_query_seq(f.handle, view, n, bm, hits)
            torch.cuda.synchronize()
            wbm, wc, n_valid = o.query_records(w.insert_bases[a:a + n], None, threads=True)
            _first_diff(bm.cpu().numpy().view(np.uint32), wbm, "chunk-mode bitmap words (n = %d)" % n)
            assert int(hits.item()) == int(wc.sum()) == n_valid
    o.close()


def test_strided_chunk_fallback_behind_record_mode():
    """A batch of 150-base reads plus ONE record above the record-mode limit hands the whole batch to the chunk-mode
    query kernel, which then runs with a capped grid and STRIDES over several chunks per thread (> 4.85 M symbols):
    the staging slots are reused from one chunk to the next."""
    w = _config3()
    n_reads = 60_000
    reads = w.read_batch(0, n_reads)                               # 9 M symbols
    lens = np.full(n_reads + 1, 150, dtype=np.int64)
    lens[30_000] = 5000
    offs = np.concatenate(([0], np.cumsum(lens))).astype(np.uint64)
    q = np.empty(int(offs[-1]), dtype=np.uint8)
    a = 30_000 * 150
    q[:a] = reads[:a]
    q[a:a + 5000] = w.insert_bases[1_000_000:1_005_000]
    q[a + 5000:] = reads[a:]
    ins = np.ascontiguousarray(w.insert_bases[:20_000_000])
    o = oracle.OracleSBF(num_bits=1 << 30, **DEFAULT)
    o.insert_records(ins, threads=True)
    with sbf.SuperBloomFilter(num_bits=1 << 30, **DEFAULT) as f:
        f.insert_seq(_dev(ins))
        for rep in range(3):                                       # an ordering bug would be intermittent
            bm = torch.full(((q.size + 31) // 32,), -1, dtype=torch.int32, device="cuda")
            hc = torch.full((offs.size - 1,), -1, dtype=torch.int32, device="cuda")
            f.query_records(_dev(q), _dev(offs.view(np.int64)), bm, hc)
            torch.cuda.synchronize()
            if rep == 0:
                wbm, wc, _ = o.query_records(q, offs, threads=True)
            _first_diff(bm.cpu().numpy().view(np.uint32), wbm, "bitmap words")
            _first_diff(hc.cpu().numpy().view(np.uint32), wc, "hit counts")
    o.close()


AXES = sorted({(s, 16, 4) for s in seqgen.SWEEP_S} | {(28, m, 4) for m in seqgen.SWEEP_M} | {(28, 16, h) for h in seqgen.SWEEP_H})


@pytest.mark.parametrize("s,m,H", AXES)
def test_config5_axes_at_full_config3_size(s, m, H):
    """BASELINE config 5, the one-factor-at-a-time axes through (28,16,4) at FULL size: the whole
    250 Mbp sequence into a 2^32-bit filter (every filter byte) and one batch of 10^6 reads (bitmap + counts)."""
    w = _config3()
    params = dict(k=31, m=m, s=s, H=H)
    nb = w.params["num_bits"]
    n_reads = 1_000_000
    if "reads" not in _c3:
        _c3["reads"] = w.read_batch(0, n_reads)
    reads, offs = _c3["reads"], seqgen.fixed_offsets(n_reads, w.read_len)
    o = oracle.OracleSBF(num_bits=nb, **params)
    o.insert_records(w.insert_bases, threads=True)
    with sbf.SuperBloomFilter(num_bits=nb, **params) as f:
        assert f.specialized
        f.insert_seq(_dev(w.insert_bases))
        torch.cuda.synchronize()
        _first_diff(f.export_bits(), o.export_bits(), "filter bytes %r" % (params,))
        bm = torch.full(((reads.size + 31) // 32,), -1, dtype=torch.int32, device="cuda")
        hc = torch.full((n_reads,), -1, dtype=torch.int32, device="cuda")
        f.query_records(_dev(reads), _dev(offs.view(np.int64)), bm, hc)
        torch.cuda.synchronize()
        wbm, wc, _ = o.query_records(reads, offs, threads=True)
        _first_diff(bm.cpu().numpy().view(np.uint32), wbm, "bitmap words %r" % (params,))
        _first_diff(hc.cpu().numpy().view(np.uint32), wc, "hit counts %r" % (params,))
    o.close()


@pytest.mark.parametrize("log2_bits", seqgen.SWEEP_LOG2_BITS)
def test_config5_filter_sizes_at_full_config3_size(log2_bits):
    """BASELINE config 5's seven filter sizes 2^28 .. 2^34 bits at (28,16,4): full sequence, one batch of 10^6 reads."""
    if log2_bits == 32:
        pytest.skip("2^32 bits is test_config3_full_size_filter_bitmap_counts")
    w = _config3()
    nb = 1 << log2_bits
    n_reads = 1_000_000
    if "reads" not in _c3:
        _c3["reads"] = w.read_batch(0, n_reads)
    reads, offs = _c3["reads"], seqgen.fixed_offsets(n_reads, w.read_len)
    o = oracle.OracleSBF(num_bits=nb, **DEFAULT)
    o.insert_records(w.insert_bases, threads=True)
    with sbf.SuperBloomFilter(num_bits=nb, **DEFAULT) as f:
        assert f.num_shards == o.num_shards == 1 << (log2_bits - 8)
        f.insert_seq(_dev(w.insert_bases))
        torch.cuda.synchronize()
        _first_diff(f.export_bits(), o.words().reshape(-1).view(np.uint8), "filter bytes at 2^%d bits" % log2_bits)
        bm = torch.full(((reads.size + 31) // 32,), -1, dtype=torch.int32, device="cuda")
        hc = torch.full((n_reads,), -1, dtype=torch.int32, device="cuda")
        f.query_records(_dev(reads), _dev(offs.view(np.int64)), bm, hc)
        torch.cuda.synchronize()
        wbm, wc, _ = o.query_records(reads, offs, threads=True)
        _first_diff(bm.cpu().numpy().view(np.uint32), wbm, "bitmap words at 2^%d bits" % log2_bits)
        _first_diff(hc.cpu().numpy().view(np.uint32), wc, "hit counts at 2^%d bits" % log2_bits)
    o.close()

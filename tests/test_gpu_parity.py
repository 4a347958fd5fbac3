"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, bit for bit, on the same
seeded inputs.  Filter words after insert, the result bitmap and the hit counts are integer work,
so the bar is exact equality (north_star).  Run with -m gpu on the B200 box."""
import numpy as np
import pytest

import oracle
import seqgen
import paper_2606_24417_b200 as sbf

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

DEFAULT = dict(k=31, m=16, s=28, H=4)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_insert(f, bases, offsets=None, stream=None):
    d = dev(bases)
    if offsets is None:
        sbf.sbf_insert_seq(f.handle, d, d.numel(), stream)
    else:
        o = dev(offsets.astype(np.uint64).view(np.int64))
        sbf.sbf_insert_records(f.handle, d, o, offsets.size - 1, d.numel(), stream)
    torch.cuda.synchronize()


def gpu_query(f, bases, offsets=None, counts=True):
    d = dev(bases)
    n = d.numel()
    bm = torch.full(((n + 31) // 32,), -1, dtype=torch.int32, device="cuda")  # poisoned: every word must be written
    if offsets is None:
        hits = torch.full((1,), -1, dtype=torch.int64, device="cuda") if counts else None
        sbf.sbf_query_seq(f.handle, d, n, bm, hits)
        torch.cuda.synchronize()
        return bm.cpu().numpy().view(np.uint32), (int(hits.item()) if counts else None)
    o = dev(offsets.astype(np.uint64).view(np.int64))
    hc = torch.full((offsets.size - 1,), -1, dtype=torch.int32, device="cuda") if counts else None
    sbf.sbf_query_records(f.handle, d, o, offsets.size - 1, n, bm, hc)
    torch.cuda.synchronize()
    return bm.cpu().numpy().view(np.uint32), (hc.cpu().numpy().view(np.uint32) if counts else None)


def check_parity(params, num_bits, ins_bases, ins_offsets, q_bases, q_offsets, expect_specialized=None):
    o = oracle.OracleSBF(num_bits=num_bits, **params)
    o.insert_records(ins_bases, ins_offsets, threads=True)
    with sbf.SuperBloomFilter(num_bits=num_bits, **params) as f:
        if expect_specialized is not None:
            assert f.specialized == expect_specialized
        assert f.num_shards == o.num_shards
        gpu_insert(f, ins_bases, ins_offsets)
        got = f.export_bits()
        want = o.export_bits()
        assert got.size == want.size
        if not np.array_equal(got, want):
            bad = np.flatnonzero(got != want)
            raise AssertionError("filter differs in %d bytes of %d, first at byte %d (shard %d)" %
                                 (bad.size, got.size, bad[0], bad[0] // 32))
        for qb, qo in ((q_bases, q_offsets), (ins_bases, ins_offsets)):
            if qb is None:
                continue
            bm, hc = gpu_query(f, qb, qo)
            wbm, wcounts, _ = o.query_records(qb, qo, threads=True)
            if not np.array_equal(bm, wbm):
                bad = np.flatnonzero(bm != wbm)
                raise AssertionError("bitmap differs in %d words of %d, first word %d: got %08x want %08x" %
                                     (bad.size, bm.size, bad[0], bm[bad[0]], wbm[bad[0]]))
            if qo is None:
                assert hc == int(wcounts.sum())
            else:
                assert np.array_equal(hc, wcounts)
    o.close()


# ------------------------------------------------------------------------------------------------
def test_config1_tiny_full():
    """BASELINE config 1 at full size: filter bytes, all-true self query, alien bitmap."""
    w = seqgen.config1()
    check_parity(DEFAULT, w.params["num_bits"], w.insert_bases, None, w.extra["alien"], None, expect_specialized=True)


def test_config1_self_query_all_true():
    w = seqgen.config1()
    with sbf.SuperBloomFilter(num_bits=1 << 24, **DEFAULT) as f:
        gpu_insert(f, w.insert_bases)
        bm, hits = gpu_query(f, w.insert_bases)
        n = w.insert_bases.size
        bits = oracle.bitmap_bits(bm, n)
        assert bits[: n - 30].all() and not bits[n - 30:].any()
        assert hits == n - 30


def test_config2_reduced_records_and_reads():
    """Config 2 shape at 1/10 scale: Markov + repeats, reads half sampled / half random, per-read counts."""
    w = seqgen.config2(scale=0.1)
    reads = w.read_batch(0, 20000)
    offs = seqgen.fixed_offsets(20000, 150)
    check_parity(DEFAULT, 1 << 24, w.insert_bases, None, reads, offs)


def test_config3_shape_with_n_runs():
    """Config 3 shape at reduced scale: order-5 Markov with N runs; reads overlapping N."""
    w = seqgen.config3(scale=0.01)
    reads = w.read_batch(0, 30000)
    offs = seqgen.fixed_offsets(30000, 150)
    check_parity(DEFAULT, 1 << 26, w.insert_bases, None, reads, offs)


def test_config4_shape_multi_record_insert():
    """Config 4 shape at reduced scale: 24 records inserted as one dense batch."""
    w = seqgen.config4(scale=0.001)
    reads = w.read_batch(0, 10000)
    offs = seqgen.fixed_offsets(10000, 150)
    check_parity(DEFAULT, 1 << 27, w.insert_bases, w.insert_offsets, reads, offs)


SWEEP_AXES = sorted({(s, 16, 4) for s in seqgen.SWEEP_S} | {(28, m, 4) for m in seqgen.SWEEP_M} |
                    {(28, 16, h) for h in seqgen.SWEEP_H})


@pytest.mark.parametrize("s,m,H", SWEEP_AXES)
def test_config5_axes_specialized(s, m, H):
    w = seqgen.config3(scale=0.002)
    reads = w.read_batch(0, 4000)
    offs = seqgen.fixed_offsets(4000, 150)
    check_parity(dict(k=31, m=m, s=s, H=H), 1 << 22, w.insert_bases, None, reads, offs, expect_specialized=True)


@pytest.mark.parametrize("s,m,H", [(24, 12, 8), (26, 20, 1), (30, 14, 6), (31, 18, 2), (24, 20, 6), (31, 12, 1), (26, 14, 8)])
def test_config5_cross_product_specialized(s, m, H):
    """Off-axis points of the 125-point cross product also have specialised instances (sbf_inst_sweep.cu)."""
    w = seqgen.config3(scale=0.001)
    reads = w.read_batch(0, 2000)
    offs = seqgen.fixed_offsets(2000, 150)
    check_parity(dict(k=31, m=m, s=s, H=H), 1 << 21, w.insert_bases, None, reads, offs, expect_specialized=True)
    check_parity(dict(k=31, m=m, s=s, H=H), 1 << 21, w.insert_bases, None, reads[:150 * 700], None, expect_specialized=True)


@pytest.mark.parametrize("s,m,H", [(27, 8, 4), (28, 16, 12), (28, 16, 16), (16, 4, 4), (31, 31, 4), (25, 16, 4)])
def test_parameters_outside_the_tables_run_the_runtime_kernel(s, m, H):
    """Any other legal (k,m,s,H), and H > 10 (A6), runs the runtime-parameter kernel: same bits."""
    w = seqgen.config3(scale=0.001)
    reads = w.read_batch(0, 2000)
    offs = seqgen.fixed_offsets(2000, 150)
    check_parity(dict(k=31, m=m, s=s, H=H), 1 << 21, w.insert_bases, None, reads, offs, expect_specialized=False)


@pytest.mark.parametrize("k,m,s,H", [(9, 5, 6, 4), (32, 16, 28, 4), (21, 11, 21, 3), (15, 15, 12, 5),
                                     (1, 1, 1, 1), (2, 1, 2, 2), (32, 32, 32, 4), (17, 3, 9, 7)])
def test_other_k(k, m, s, H):
    rng = np.random.default_rng(k * 1000 + m)
    seq = seqgen.uniform(100 + k, 60000)
    seq[rng.integers(0, seq.size, 40)] = ord("N")
    seq[5000:5100] = ord("n")
    seq[7000:7003] = np.frombuffer(b"acg", dtype=np.uint8)
    q = seqgen.uniform(200 + k, 50000)
    q[:20000] = seq[10000:30000]
    check_parity(dict(k=k, m=m, s=s, H=H), 1 << 16, seq, None, q, None)


# ------------------------------------------------------------------------------------------------ edge cases
def _ragged_records(seed, n_rec, max_len):
    rng = np.random.default_rng(seed)
    lens = rng.integers(0, max_len, n_rec)
    lens[rng.integers(0, n_rec, n_rec // 10)] = 0            # empty records
    lens[rng.integers(0, n_rec, n_rec // 10)] = 30           # k-1: no k-mer
    lens[rng.integers(0, n_rec, n_rec // 10)] = 31           # exactly one k-mer
    offs = np.concatenate(([0], np.cumsum(lens))).astype(np.uint64)
    bases = seqgen.uniform(seed, int(offs[-1]))
    return bases, offs


def test_ragged_and_empty_records():
    bases, offs = _ragged_records(7, 3000, 400)
    qb, qo = _ragged_records(8, 2000, 300)
    qb[:5000] = bases[:5000]
    check_parity(DEFAULT, 1 << 20, bases, offs, qb, qo)


def test_records_vs_concatenation_differ_only_at_boundaries():
    """No k-mer spans two records: inserting as records sets a subset of the bits of the concatenation."""
    bases, offs = _ragged_records(9, 500, 300)
    with sbf.SuperBloomFilter(num_bits=1 << 22, **DEFAULT) as f:
        gpu_insert(f, bases, offs)
        a = f.export_bits()
        f.clear()
        gpu_insert(f, bases, None)
        b = f.export_bits()
    assert np.array_equal(a & b, a) and not np.array_equal(a, b)


@pytest.mark.parametrize("n", [0, 1, 30, 31, 32, 127, 128, 129, 4095, 4096 + 31])
def test_tiny_lengths(n):
    seq = seqgen.uniform(11, max(n, 1))[:n]
    o = oracle.OracleSBF(num_bits=1 << 14, **DEFAULT)
    o.insert_records(seq)
    with sbf.SuperBloomFilter(num_bits=1 << 14, **DEFAULT) as f:
        if n:
            gpu_insert(f, seq)
            assert np.array_equal(f.export_bits(), o.export_bits())
            bm, hits = gpu_query(f, seq)
            wbm, wc, _ = o.query_records(seq)
            assert np.array_equal(bm, wbm) and hits == int(wc.sum()) == max(0, n - 30)
        else:
            sbf.sbf_insert_seq(f.handle, None, 0)
            sbf.sbf_query_seq(f.handle, None, 0, None, None)
            assert not f.export_bits().any()


def test_all_invalid_and_low_complexity():
    n = 20000
    for seq in (np.full(n, ord("N"), np.uint8), np.full(n, ord("A"), np.uint8),
                np.frombuffer((b"AC" * (n // 2)), dtype=np.uint8).copy(),
                np.frombuffer((b"ACGTTGCA" * (n // 8)), dtype=np.uint8).copy()):
        check_parity(DEFAULT, 1 << 16, seq, None, seqgen.uniform(5, 5000), None)


def test_unaligned_device_pointer():
    """d_seq need not be 16-byte aligned: views at byte offsets 1..15 give the same bits."""
    seq = seqgen.uniform(21, 50000)
    o = oracle.OracleSBF(num_bits=1 << 18, **DEFAULT)
    for shift in (1, 3, 8, 15):
        o.clear()
        o.insert_records(seq[shift:])
        with sbf.SuperBloomFilter(num_bits=1 << 18, **DEFAULT) as f:
            d = dev(seq)
            view = d[shift:]
            sbf.sbf_insert_seq(f.handle, view.data_ptr(), view.numel())
            torch.cuda.synchronize()
            assert np.array_equal(f.export_bits(), o.export_bits())


def test_order_independence_and_idempotence_on_gpu():
    """P6 on the device: permuting the records or inserting twice leaves identical bytes (atomics race test)."""
    bases, offs = _ragged_records(13, 2000, 500)
    lens = np.diff(offs.astype(np.int64))
    perm = np.random.default_rng(1).permutation(lens.size)
    pb = np.concatenate([bases[int(offs[i]):int(offs[i + 1])] for i in perm] + [np.zeros(0, np.uint8)])
    po = np.concatenate(([0], np.cumsum(lens[perm]))).astype(np.uint64)
    with sbf.SuperBloomFilter(num_bits=1 << 20, **DEFAULT) as f:
        gpu_insert(f, bases, offs)
        a = f.export_bits()
        gpu_insert(f, bases, offs)
        assert np.array_equal(a, f.export_bits())
        f.clear()
        gpu_insert(f, pb, po)
        assert np.array_equal(a, f.export_bits())


def test_streams_and_reserve():
    seq = seqgen.uniform(31, 300000)
    o = oracle.OracleSBF(num_bits=1 << 22, **DEFAULT)
    o.insert_records(seq, threads=True)
    st = torch.cuda.Stream()
    with sbf.SuperBloomFilter(num_bits=1 << 22, **DEFAULT) as f:
        f.reserve(seq.size)
        d = dev(seq)
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            sbf.sbf_insert_seq(f.handle, d, d.numel(), st)
        st.synchronize()
        assert np.array_equal(f.export_bits(), o.export_bits())


def test_import_export_or_roundtrip():
    a = seqgen.uniform(41, 100000)
    b = seqgen.uniform(42, 100000)
    o = oracle.OracleSBF(num_bits=1 << 20, **DEFAULT)
    o.insert_records(a)
    o.insert_records(b)
    with sbf.SuperBloomFilter(num_bits=1 << 20, **DEFAULT) as fa, sbf.SuperBloomFilter(num_bits=1 << 20, **DEFAULT) as fb:
        gpu_insert(fa, a)
        gpu_insert(fb, b)
        sbf.sbf_or_bits_device(fa.handle, sbf.sbf_filter_device_ptr(fb.handle), fa.num_shards * 32)
        torch.cuda.synchronize()
        merged = fa.export_bits()
        assert np.array_equal(merged, o.export_bits())
        fb.import_bits(merged)
        assert np.array_equal(fb.export_bits(), merged)


@pytest.mark.parametrize("world,window", [(2, 1 << 28), (3, 40_000), (5, 9_999)])
def test_replica_merge_on_one_device(world, window):
    """The multi-GPU exchange's plan and kernels on ONE device: `world` replicas filled from a partition of the batch,
    merged with replicas.merge_local_replicas (sbf_or_peers_range_device per slice, then the gather copies) — every
    replica must equal the oracle's single filter.  Windows smaller than the filter, a ragged last window, slices of
    unequal length."""
    from paper_2606_24417_b200 import replicas
    seq = seqgen.markov(31, 5, 0.41, 400_000)
    seq[100_000:100_300] = ord("N")
    o = oracle.OracleSBF(num_bits=1 << 21, **DEFAULT)
    o.insert_records(seq, threads=True)
    fs = [sbf.SuperBloomFilter(num_bits=1 << 21, **DEFAULT) for _ in range(world)]
    try:
        for r, f in enumerate(fs):
            a, e = replicas.partition_positions(seq.size, DEFAULT["k"], world, r)
            gpu_insert(f, seq[a:e])
        n = replicas.merge_local_replicas([f.handle for f in fs], window_bytes=window)
        torch.cuda.synchronize()
        assert n >= world
        want = o.export_bits()
        for r, f in enumerate(fs):
            assert np.array_equal(f.export_bits(), want), "replica %d differs from the single-rank filter" % r
    finally:
        for f in fs:
            f.close()
    o.close()


def test_host_facing_calls_match_device_facing():
    """The host-facing forms (chunked staging) give the same filter, bitmap and counts."""
    w = seqgen.config2(scale=0.05)
    reads = w.read_batch(0, 5000)
    offs = seqgen.fixed_offsets(5000, 150)
    o = oracle.OracleSBF(num_bits=1 << 23, **DEFAULT)
    o.insert_records(w.insert_bases, threads=True)
    wbm, wcounts, _ = o.query_records(reads, offs, threads=True)
    with sbf.SuperBloomFilter(num_bits=1 << 23, **DEFAULT) as f:
        sbf.sbf_insert_seq_host(f.handle, w.insert_bases, w.insert_bases.size)
        assert np.array_equal(f.export_bits(), o.export_bits())
        bm = np.full((reads.size + 31) // 32, 0xFFFFFFFF, dtype=np.uint32)
        hc = np.full(5000, 0xFFFFFFFF, dtype=np.uint32)
        sbf.sbf_query_records_host(f.handle, reads, offs, 5000, bm, hc)
        assert np.array_equal(bm, wbm) and np.array_equal(hc, wcounts)
        # pinned caller memory takes the direct path
        pinned = torch.from_numpy(reads).pin_memory()
        bm2 = np.zeros_like(bm)
        hits = np.zeros(1, dtype=np.uint64)
        sbf.sbf_query_seq_host(f.handle, pinned, pinned.numel(), bm2, hits)
        wbm2, wc2, _ = o.query_records(reads, None, threads=True)
        assert np.array_equal(bm2, wbm2) and int(hits[0]) == int(wc2.sum())


def test_pack_kernel_words_and_mask():
    """a1 on its own: packed 2-bit words and the k-mer validity bits V against a plain numpy restatement."""
    rng = np.random.default_rng(3)
    seq = seqgen.uniform(51, 5000)
    seq[rng.integers(0, seq.size, 60)] = ord("N")
    seq[100:110] = np.frombuffer(b"acgtacgtXa", dtype=np.uint8)
    k = 31
    nw = (seq.size + 15) // 16
    words, mask = sbf.sbf_bench_pack(dev(seq), seq.size, k, nw)      # pack_kernel as the insert / query calls launch it
    code = np.full(256, -1, dtype=np.int64)
    for ch, v in zip(b"ACGTacgt", [0, 1, 2, 3] * 2):
        code[ch] = v
    c = code[seq]
    inv = np.concatenate((c < 0, np.ones(16 * nw + 1 - seq.size, bool)))
    cc = np.concatenate((np.where(c < 0, 0, c), np.zeros(16 * nw - seq.size, np.int64))).reshape(nw, 16)
    want_valid_words = np.zeros(nw, dtype=np.uint64)
    for j in range(16):
        want_valid_words |= cc[:, j].astype(np.uint64) << np.uint64(30 - 2 * j)
    ok_word = ~inv[: 16 * nw].reshape(nw, 16).any(axis=1)
    assert np.array_equal(words[ok_word], want_valid_words[ok_word].astype(np.uint32))
    # V[j] = some symbol of [j, j+k) is not ACGT or lies past the end: no valid k-mer starts at j
    ext = np.concatenate((inv, np.ones(k, bool)))
    cs = np.concatenate(([0], np.cumsum(ext)))
    V = (cs[k:k + 16 * nw] - cs[:16 * nw]) > 0
    want_mask = (V.reshape(nw, 16) << np.arange(16)).sum(axis=1).astype(np.uint16)
    assert np.array_equal(mask, want_mask)


def test_every_byte_value_as_a_symbol():
    """A9: ACGT in either case are the only valid symbols; every other byte value resets the window."""
    rng = np.random.default_rng(11)
    seq = seqgen.uniform(12, 400_000)
    lower = rng.random(seq.size) < 0.3
    seq[lower] |= 0x20                                   # lower-case a c g t are valid too
    pos = rng.choice(seq.size, 256 * 8, replace=False)   # every byte value, 8 times, far enough apart
    seq[pos] = np.tile(np.arange(256, dtype=np.uint8), 8)
    q = seqgen.uniform(13, 100_000)
    q[rng.choice(q.size, 512, replace=False)] = np.tile(np.arange(256, dtype=np.uint8), 2)
    check_parity(DEFAULT, 1 << 24, seq, None, q, None, True)


def test_record_mode_and_its_device_side_fallback():
    """Short records run one-thread-per-record (stream_rec_kernel); one record above the limit makes the
    device-side flag hand the whole batch to the chunk kernels.  Both must give the oracle's bits."""
    seq = seqgen.markov(31, 5, 0.41, 600_000)
    seq[1000:1100] = ord("N")
    rng = np.random.default_rng(5)
    # (a) ragged short records incl. empty ones, lengths 0..400, every start alignment
    lens = rng.integers(0, 400, size=2500)
    lens[::97] = 0
    lens[5] = 30; lens[6] = 31; lens[7] = 32; lens[8] = 1
    offs = np.concatenate(([0], np.cumsum(lens))).astype(np.uint64)
    q = seqgen.reads(9, seq, 0, (int(offs[-1]) + 149) // 150, 150, 0.01)[:int(offs[-1])].copy()
    q[rng.choice(q.size, 300, replace=False)] = ord("N")
    check_parity(DEFAULT, 1 << 24, seq, None, q, offs, True)
    # (b) same mean length, but one record of 5000 symbols (> 1024): chunk kernels take over
    lens2 = lens.copy(); lens2[100] = 5000
    offs2 = np.concatenate(([0], np.cumsum(lens2))).astype(np.uint64)
    q2 = seqgen.reads(10, seq, 0, (int(offs2[-1]) + 149) // 150, 150, 0.01)[:int(offs2[-1])].copy()
    check_parity(DEFAULT, 1 << 24, seq, None, q2, offs2, True)
    # (c) fixed 150-base reads whose count is not a multiple of the CTA size, other k / H
    for params in (dict(k=21, m=11, s=21, H=3), dict(k=31, m=16, s=28, H=8), dict(k=9, m=5, s=6, H=4)):
        n = 1237
        qq = seqgen.reads(11, seq, 0, n, 150, 0.02)
        check_parity(params, 1 << 22, seq[:200_000], None, qq, seqgen.fixed_offsets(n, 150), True)

"""GPU parity of the FASTA / FASTQ host path (sbf_insert_fastx_host / sbf_query_fastx_host): the raw
text is chunked, copied and normalised ON THE DEVICE, then inserted / queried as a dense record batch.  Expected values
come from the oracle side only: oracle/fastx.py reads the same text line by line, the oracle inserts / queries the dense
batch it yields.  Small chunks put chunk edges inside header lines, sequence lines, quality lines, line ends ("\\r\\n"
split across two chunks), records and k-mers; one case runs the default 32 Mi chunks on a 75 MB genome-like text."""
import string

import numpy as np
import pytest

import oracle
from oracle import fastx
import seqgen
import paper_2606_24417_b200 as sbf

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

DEFAULT = dict(k=31, m=16, s=28, H=4)


def _records(seed, n, max_len, alphabet=0):
    rng = np.random.default_rng(seed)
    lens = rng.integers(0, max_len, n)
    lens[rng.integers(0, n, max(1, n // 8))] = 0
    lens[rng.integers(0, n, max(1, n // 8))] = 30
    out = []
    for i, l in enumerate(lens):
        r = seqgen.uniform(seed * 1000 + i, int(l))
        if alphabet == oracle.PROTEIN:
            r = np.frombuffer(string.ascii_uppercase.encode(), dtype=np.uint8)[(r.astype(np.int64) * 7 + np.arange(r.size)) % 26].copy()
        if l > 40 and i % 5 == 0:
            r[int(l) // 2] = ord("N") if alphabet != oracle.PROTEIN else ord("*")
        out.append(r)
    return out


def _check_insert(params, alphabet, text, chunk, num_bits=1 << 22, fmt=0):
    bases, offs = fastx.dense(text, fmt)
    o = oracle.OracleSBF(num_bits=num_bits, alphabet=alphabet, **params)
    o.insert_records(bases, offs, threads=True)
    n_rec_want = len(fastx.parse(text, fmt)[1])
    with sbf.SuperBloomFilter(num_bits=num_bits, alphabet=alphabet, **params) as f:
        if chunk:
            sbf.sbf_set_host_chunk(f.handle, chunk)
        n_rec, n_bases = sbf.sbf_insert_fastx_host(f.handle, text, len(text), fmt)
        assert (n_rec, n_bases) == (n_rec_want, bases.size)
        got, want = f.export_bits(), o.export_bits()
        assert np.array_equal(got, want), "filter differs in %d bytes (chunk %d)" % (np.count_nonzero(got != want), chunk)
    return o


def _check_query(o, params, alphabet, ins_bases, ins_offs, text, chunk, num_bits=1 << 22, fmt=0):
    bases, offs = fastx.dense(text, fmt, with_pre=False)
    _, want_counts, _ = o.query_records(bases, offs, threads=True)
    with sbf.SuperBloomFilter(num_bits=num_bits, alphabet=alphabet, **params) as f:
        d = torch.from_numpy(ins_bases).cuda()
        sbf.sbf_insert_records(f.handle, d, torch.from_numpy(ins_offs.view(np.int64)).cuda(), ins_offs.size - 1, d.numel())
        if chunk:
            sbf.sbf_set_host_chunk(f.handle, chunk)
        hc = np.full(offs.size - 1 + 3, 0xFFFFFFFF, dtype=np.uint32)
        n_rec, n_bases = sbf.sbf_query_fastx_host(f.handle, text, len(text), hc, hc.size, fmt)
        assert n_rec == offs.size - 1
        assert np.array_equal(hc[:n_rec], want_counts), "hit counts differ (chunk %d)" % chunk
        if n_rec > 1:
            with pytest.raises(sbf.SBFError):
                sbf.sbf_query_fastx_host(f.handle, text, len(text), hc, n_rec - 1, fmt)


@pytest.mark.parametrize("chunk", [1152, 4096, 0])
@pytest.mark.parametrize("crlf", [False, True])
def test_fasta_insert_and_query(chunk, crlf):
    recs = _records(3, 60, 900) + [seqgen.uniform(77, 9000)]          # one record longer than the small chunks
    text = b"ACGTTGCA" * 9 + b"\n" + seqgen.fasta_text(recs, 60, crlf)  # sequence text before the first header
    o = _check_insert(DEFAULT, 0, text, chunk)
    q_recs = [r.copy() for r in recs[::2]] + _records(4, 30, 500)
    q_text = seqgen.fasta_text(q_recs, 70, crlf)
    ins_bases, ins_offs = fastx.dense(text)
    _check_query(o, DEFAULT, 0, ins_bases, ins_offs, q_text, chunk)
    o.close()


@pytest.mark.parametrize("chunk", [1152, 2048, 0])
@pytest.mark.parametrize("crlf,final_newline", [(False, True), (True, True), (False, False)])
def test_fastq_insert_and_query(chunk, crlf, final_newline):
    genome = seqgen.markov(31, 5, 0.41, 60_000)
    reads = seqgen.reads(9, genome, 0, 400, 150, 0.01).reshape(400, 150)
    recs = [reads[i, :int(l)] for i, l in enumerate(np.random.default_rng(1).integers(0, 151, 400))]
    text = seqgen.fastq_text(recs, crlf, final_newline)
    assert fastx.detect(text) == fastx.FASTQ
    o = _check_insert(DEFAULT, 0, text, chunk)
    o.close()
    # query the reads against the genome
    o = oracle.OracleSBF(num_bits=1 << 22, **DEFAULT)
    o.insert_records(genome)
    _check_query(o, DEFAULT, 0, genome, np.array([0, genome.size], dtype=np.uint64), text, chunk)
    o.close()


@pytest.mark.parametrize("alphabet,params", [(oracle.PROTEIN, dict(k=12, m=6, s=10, H=4)), (oracle.TRIPLET, dict(k=10, m=5, s=8, H=4)),
                                             (oracle.DNA, dict(k=63, m=31, s=60, H=4))])
def test_fasta_other_alphabets_and_wide_kmers(alphabet, params):
    recs = _records(11 + alphabet, 40, 1500, alphabet)
    text = seqgen.fasta_text(recs, 61)                              # 61 columns: line ends off every 3-byte grid
    for chunk in (1152, 4096):
        o = _check_insert(params, alphabet, text, chunk, num_bits=1 << 20)
        ins_bases, ins_offs = fastx.dense(text)
        _check_query(o, params, alphabet, ins_bases, ins_offs, seqgen.fasta_text(recs[::3] + _records(5, 10, 800, alphabet), 80),
                     chunk, num_bits=1 << 20)
        o.close()


@pytest.mark.parametrize("chunk", [1152, 0])
@pytest.mark.parametrize("tail", [b"\n\n", b"\n\n\n\n", b"\r\n\r\n", b"\n\n@late\nACGTACGTACGTACGTACGTACGTACGTACGTACGT\n+\nII\n"])
def test_fastq_blank_lines_open_no_record(chunk, tail):
    """A text ending in a blank line (or holding one between records) has the records the oracle-side reader finds, no
    extra empty one (A23): the record count, the filter and the per-record hit counts agree, with max_records equal to
    the true count."""
    genome = seqgen.markov(32, 5, 0.41, 30_000)
    recs = [r for r in seqgen.reads(10, genome, 0, 60, 150, 0.01).reshape(60, 150)]
    text = seqgen.fastq_text(recs, False, final_newline=False) + tail
    n_want = len(fastx.parse(text, fastx.FASTQ)[1])
    assert n_want == 60 + (tail.count(b"II") > 0)          # the grid-shifted tail yields one (empty) record more
    for fmt in (0, fastx.FASTQ):
        o = _check_insert(DEFAULT, 0, text, chunk, fmt=fmt)
        o.close()
    o = oracle.OracleSBF(num_bits=1 << 22, **DEFAULT)
    o.insert_records(genome)
    bases, offs = fastx.dense(text, fastx.FASTQ, with_pre=False)
    _, want_counts, _ = o.query_records(bases, offs, threads=True)
    with sbf.SuperBloomFilter(num_bits=1 << 22, **DEFAULT) as f:
        d = torch.from_numpy(genome).cuda()
        sbf.sbf_insert_seq(f.handle, d, d.numel())
        if chunk:
            sbf.sbf_set_host_chunk(f.handle, chunk)
        hc = np.full(n_want, 0xFFFFFFFF, dtype=np.uint32)
        n_rec, _ = sbf.sbf_query_fastx_host(f.handle, text, len(text), hc, n_want, fastx.FASTQ)   # capacity = true count
        assert n_rec == n_want and np.array_equal(hc, want_counts)
    o.close()


def test_degenerate_texts():
    with sbf.SuperBloomFilter(num_bits=1 << 16, **DEFAULT) as f:
        for text in (b"", b"\n\n\n", b">only a header", b">h\n", b"@h\n\n+\n\n", b"ACGT", b">a\n>b\n>c\n"):
            n_rec, n_bases = sbf.sbf_insert_fastx_host(f.handle, text, len(text), 0)
            pre, recs = fastx.parse(text)
            assert n_rec == len(recs) and n_bases == len(pre) + sum(len(r) for r in recs), text
        assert not f.export_bits().any()


@pytest.mark.slow
def test_fasta_genome_default_chunks():
    """75 MB of FASTA text in three 32 Mi chunks: 6 records of 5-20 Mbp wrapped at 60 columns."""
    w = seqgen.config3(scale=0.29)
    cuts = [0, 5_000_000, 25_000_000, 25_000_001, 40_000_000, 60_000_000, w.insert_bases.size]
    recs = [w.insert_bases[a:b] for a, b in zip(cuts[:-1], cuts[1:])]
    text = seqgen.fasta_text(recs, 60)
    assert len(text) > 70 << 20
    bases, offs = fastx.dense(text)
    o = oracle.OracleSBF(num_bits=1 << 30, **DEFAULT)
    o.insert_records(bases, offs, threads=True)
    pinned = torch.from_numpy(np.frombuffer(text, dtype=np.uint8).copy()).pin_memory()
    with sbf.SuperBloomFilter(num_bits=1 << 30, **DEFAULT) as f:
        n_rec, n_bases = sbf.sbf_insert_fastx_host(f.handle, pinned, pinned.numel(), 1)
        assert (n_rec, n_bases) == (6, bases.size)
        got, want = f.export_bits(), o.export_bits()
        assert np.array_equal(got, want), "filter differs in %d bytes" % np.count_nonzero(got != want)
    o.close()

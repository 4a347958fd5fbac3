"""GPU parity of the WIDE path: DNA with 32 < k <= 64, the protein alphabet and the DNA-triplet
alphabet (readings A19-A22) through sbf_create_ex, against the oracle's wide path (pinned in
tests/test_oracle_wide_pins.py), bit for bit: filter bytes, result bitmap (indexed by byte position), hit counts.
Covers one sequence and ragged record batches (empty records, records shorter than a k-mer, lengths not a multiple of
three for triplets), invalid symbols, lower case, unaligned device pointers, the host-facing calls in several chunks
(triplet framing across chunk edges), and the edge of the 128-bit packing (k * symbol bits = 125, 126, 128)."""
import string

import numpy as np
import pytest

import oracle
import seqgen
import paper_2606_24417_b200 as sbf

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

AA = np.frombuffer(string.ascii_uppercase.encode(), dtype=np.uint8)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rand_text(alphabet, seed, n):
    if alphabet == oracle.PROTEIN:
        r = seqgen.uniform(seed, 3 * n).astype(np.int64).reshape(n, 3)
        idx = (((r[:, 0] >> 1) & 3) * 16 + ((r[:, 1] >> 1) & 3) * 4 + ((r[:, 2] >> 1) & 3)) % 26
        return AA[idx].copy()
    return seqgen.uniform(seed, n)


def ragged_offsets(rng, total, mean):
    lens, left = [], total
    while left > 0:
        l = int(min(left, rng.integers(0, 2 * mean + 1)))
        lens.append(l); left -= l
        if rng.random() < 0.05:
            lens.append(0)
    return np.concatenate(([0], np.cumsum(lens))).astype(np.uint64)


def check(alphabet, k, m, s, H, num_bits, ins, ins_offs, q, q_offs, specialized=False):
    o = oracle.OracleSBF(k, m, s, H, num_bits, alphabet=alphabet)
    n_ins = o.insert_records(ins, ins_offs, threads=True)
    assert n_ins > 0
    with sbf.SuperBloomFilter(k=k, m=m, s=s, H=H, num_bits=num_bits, alphabet=alphabet) as f:
        assert f.specialized == specialized and f.num_shards == o.num_shards
        d = dev(ins)
        if ins_offs is None:
            sbf.sbf_insert_seq(f.handle, d, d.numel())
        else:
            sbf.sbf_insert_records(f.handle, d, dev(ins_offs.view(np.int64)), ins_offs.size - 1, d.numel())
        torch.cuda.synchronize()
        got, want = f.export_bits(), o.export_bits()
        assert np.array_equal(got, want), "filter differs in %d bytes" % np.count_nonzero(got != want)
        for qb, qo in ((q, q_offs), (ins, ins_offs)):
            dq = dev(qb)
            bm = torch.full(((qb.size + 31) // 32,), -1, dtype=torch.int32, device="cuda")
            wbm, wc, _ = o.query_records(qb, qo, threads=True)
            if qo is None:
                hits = torch.full((1,), -1, dtype=torch.int64, device="cuda")
                sbf.sbf_query_seq(f.handle, dq, qb.size, bm, hits)
                torch.cuda.synchronize()
                assert int(hits.item()) == int(wc.sum())
            else:
                hc = torch.full((qo.size - 1,), -1, dtype=torch.int32, device="cuda")
                sbf.sbf_query_records(f.handle, dq, dev(qo.view(np.int64)), qo.size - 1, qb.size, bm, hc)
                torch.cuda.synchronize()
                assert np.array_equal(hc.cpu().numpy().view(np.uint32), wc)
            assert np.array_equal(bm.cpu().numpy().view(np.uint32), wbm)
    o.close()


CASES = [(oracle.DNA, 63, 30, 59, 4), (oracle.DNA, 64, 32, 64, 8), (oracle.DNA, 33, 16, 30, 12), (oracle.DNA, 47, 20, 40, 3),
         (oracle.PROTEIN, 12, 6, 10, 4), (oracle.PROTEIN, 25, 7, 20, 4), (oracle.PROTEIN, 5, 2, 3, 2),
         (oracle.TRIPLET, 10, 5, 8, 4), (oracle.TRIPLET, 21, 9, 18, 6), (oracle.TRIPLET, 1, 1, 1, 1)]


@pytest.mark.parametrize("alphabet,k,m,s,H", CASES)
def test_one_sequence_and_ragged_records(alphabet, k, m, s, H):
    rng = np.random.default_rng(1000 * alphabet + k)
    step = 3 if alphabet == oracle.TRIPLET else 1
    bad = ord("*") if alphabet == oracle.PROTEIN else ord("N")
    ins = rand_text(alphabet, 10 + k, 120_000)
    ins[rng.integers(0, ins.size, 30)] = bad
    ins[5000:5200] |= 0x20                                   # lower case is valid too (A9 / A19)
    q = rand_text(alphabet, 20 + k, 90_001)
    q[:40_000] = ins[30_000:70_000]                          # true members (frame preserved: 30 000 is a multiple of 3)
    q[rng.integers(0, q.size, 20)] = bad
    check(alphabet, k, m, s, H, 1 << 20, ins, None, q, None)
    mean = 40 * k * step
    check(alphabet, k, m, s, H, 1 << 20, ins, ragged_offsets(rng, ins.size, mean), q, ragged_offsets(rng, q.size, mean // 3 + 1))


def test_every_byte_value_as_a_protein_symbol():
    rng = np.random.default_rng(4)
    ins = rand_text(oracle.PROTEIN, 3, 60_000)
    pos = rng.choice(ins.size, 256 * 4, replace=False)
    ins[pos] = np.tile(np.arange(256, dtype=np.uint8), 4)
    check(oracle.PROTEIN, 12, 6, 10, 4, 1 << 18, ins, None, rand_text(oracle.PROTEIN, 5, 20_000), None)


def test_unaligned_pointers_and_tiny_inputs():
    k, m, s, H = 63, 31, 60, 4
    seq = seqgen.uniform(7, 5000)
    o = oracle.OracleSBF(k, m, s, H, 1 << 16)
    with sbf.SuperBloomFilter(k=k, m=m, s=s, H=H, num_bits=1 << 16) as f:
        buf = dev(np.concatenate((np.zeros(5, np.uint8), seq)))
        for n in (0, 1, 62, 63, 64, 200, 4999):
            o.clear(); f.clear()
            view = buf[5:5 + n]
            sbf.sbf_insert_seq(f.handle, view.data_ptr() if n else None, n)
            o.insert_records(seq[:n])
            torch.cuda.synchronize()
            assert np.array_equal(f.export_bits(), o.export_bits()), n
            if n:
                bm = torch.full(((n + 31) // 32,), -1, dtype=torch.int32, device="cuda")
                sbf.sbf_query_seq(f.handle, view.data_ptr(), n, bm, None)
                torch.cuda.synchronize()
                assert np.array_equal(bm.cpu().numpy().view(np.uint32), o.query_records(seq[:n])[0])
    o.close()


@pytest.mark.parametrize("alphabet,k,m,s,H", [(oracle.PROTEIN, 12, 6, 10, 4), (oracle.TRIPLET, 7, 3, 5, 4)])
def test_more_record_boundaries_than_a_tile_lists(alphabet, k, m, s, H):
    """wide_tile_kernel lists the record boundaries of its 1 KiB tile in shared memory; a tile crossed by thousands of
    empty records overflows that list and must fall back to looking records up in the global offsets.  Also: records of
    1-3 bytes (hundreds of boundaries per tile, none of them holding a k-mer) next to ordinary ones."""
    rng = np.random.default_rng(77)
    n = 40_000
    text = rand_text(alphabet, 61, n)
    text[rng.integers(0, n, 40)] = ord("#")
    lens = []
    left = n
    while left > 0:
        r = rng.random()
        if r < 0.02:
            lens.extend([0] * int(rng.integers(1200, 3000)))      # a burst of empty records at one position
        l = int(min(left, rng.integers(1, 4) if r < 0.3 else rng.integers(20, 400)))
        lens.append(l); left -= l
    offs = np.concatenate(([0], np.cumsum(lens))).astype(np.uint64)
    assert offs[-1] == n
    check(alphabet, k, m, s, H, 1 << 18, text, offs, text[::-1].copy(), offs)


@pytest.mark.parametrize("alphabet,k,m,s,H", [(oracle.TRIPLET, 10, 5, 8, 4), (oracle.DNA, 63, 31, 60, 4), (oracle.PROTEIN, 25, 7, 20, 4)])
def test_host_facing_calls_in_several_chunks(alphabet, k, m, s, H):
    """Chunks of 1152 / 2048 bytes: k-mers straddle chunk edges (overlap k * bytes-per-symbol - 1) and, for triplets,
    the 3-byte grid of a record must be carried across edges that are not multiples of 3 from the record start."""
    rng = np.random.default_rng(k)
    total = 25_000
    ins = rand_text(alphabet, 31 + k, total)
    q = rand_text(alphabet, 32 + k, total); q[:9000] = ins[3000:12000]
    for chunk in (1152, 2048):
        ins_offs = ragged_offsets(rng, total, 700)
        q_offs = ragged_offsets(rng, total, 500)
        o = oracle.OracleSBF(k, m, s, H, 1 << 18, alphabet=alphabet)
        o_seq = oracle.OracleSBF(k, m, s, H, 1 << 18, alphabet=alphabet)
        o.insert_records(ins, ins_offs)
        o_seq.insert_records(ins)
        with sbf.SuperBloomFilter(k=k, m=m, s=s, H=H, num_bits=1 << 18, alphabet=alphabet) as f:
            sbf.sbf_set_host_chunk(f.handle, chunk)
            sbf.sbf_insert_seq_host(f.handle, ins, ins.size)
            assert np.array_equal(f.export_bits(), o_seq.export_bits())
            f.clear()
            sbf.sbf_insert_records_host(f.handle, ins, ins_offs, ins_offs.size - 1)
            assert np.array_equal(f.export_bits(), o.export_bits())
            bm = np.full((total + 31) // 32, 0xFFFFFFFF, dtype=np.uint32)
            hc = np.full(q_offs.size - 1, 0xFFFFFFFF, dtype=np.uint32)
            sbf.sbf_query_records_host(f.handle, q, q_offs, q_offs.size - 1, bm, hc)
            wbm, wc, _ = o.query_records(q, q_offs)
            assert np.array_equal(bm, wbm) and np.array_equal(hc, wc)
            bm2 = np.full_like(bm, 0xFFFFFFFF)
            hits = np.zeros(1, dtype=np.uint64)
            sbf.sbf_query_seq_host(f.handle, q, total, bm2, hits)
            wbm2, wc2, _ = o.query_records(q, None)
            assert np.array_equal(bm2, wbm2) and int(hits[0]) == int(wc2.sum())
        o.close(); o_seq.close()


# DNA k-mers of 33..64 bases that have SPECIALISED streaming instances (csrc/sbf_inst_wide.cu): the thread-serial kernels
# with a wider register window and folded (A21) m-mers / s-mers
WIDE_SPECIALISED = [(63, 31, 60, 4), (51, 25, 48, 4), (63, 40, 60, 4), (51, 31, 48, 4), (47, 24, 44, 4), (33, 16, 30, 4), (64, 41, 64, 8)]


@pytest.mark.parametrize("k,m,s,H", WIDE_SPECIALISED)
def test_specialised_wide_k_instances(k, m, s, H):
    """Insert (sequence: chunk mode; record batch: chunk mode + record-end marking with k-1 up to 63 bits), record-mode
    query of 150-base reads, its fallback (one long record), chunk-mode query of a sequence — against the oracle's wide path."""
    rng = np.random.default_rng(k)
    w = seqgen.config3(scale=0.004)                                   # 1 Mbp with an N run
    ins = w.insert_bases
    ins[rng.integers(0, ins.size, 40)] = ord("N")
    ins[7000:7400] |= 0x20
    reads = w.read_batch(0, 6000)
    offs = seqgen.fixed_offsets(6000, 150)
    check(oracle.DNA, k, m, s, H, 1 << 24, ins, None, reads, offs, specialized=True)                  # record mode
    lens = np.full(6000, 150, dtype=np.int64); lens[17] = 3000; lens[100:140] = rng.integers(0, 80, 40)
    roffs = np.concatenate(([0], np.cumsum(lens))).astype(np.uint64)
    q2 = np.concatenate((reads, seqgen.uniform(5, int(roffs[-1]) - reads.size))) if int(roffs[-1]) > reads.size else reads[:int(roffs[-1])].copy()
    check(oracle.DNA, k, m, s, H, 1 << 24, ins, ragged_offsets(rng, ins.size, 4000), q2, roffs, specialized=True)  # fallback
    check(oracle.DNA, k, m, s, H, 1 << 24, ins, None, reads, None, specialized=True)                  # chunk-mode query


@pytest.mark.slow
def test_specialised_k63_at_25_mbp():
    k, m, s, H = 63, 40, 60, 4
    w = seqgen.config3(scale=0.1)
    reads = w.read_batch(0, 200_000)
    check(oracle.DNA, k, m, s, H, 1 << 30, w.insert_bases, None, reads, seqgen.fixed_offsets(200_000, 150), specialized=True)

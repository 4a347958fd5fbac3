"""Pins of the oracle's WIDE path (other alphabets; packed k-mers wider than 64 bits, P:153 / P:435; readings
A19-A22 of DESIGN.md §3) against what does not depend on it: the already pinned narrow path (DNA, k <= 32 run through
the wide functions must give the same bytes), big-int vectors written by tests/golden/make_wide_vectors.py, plain
string manipulation, brute force on tiny inputs, invariants and the closed forms of the paper (P:86 density, Eq. (1)/(2)
per shard).  None of them compares the wide path with itself or with the CUDA path."""
import os
import string

import numpy as np
import pytest

import oracle
import seqgen

GOLD = os.path.join(os.path.dirname(__file__), "golden")
M64 = (1 << 64) - 1
AA = string.ascii_uppercase                    # the 26 protein symbols, code = index (A19)


def pack_syms(codes, bits):
    v = 0
    for c in codes:
        v = (v << bits) | c
    return v


def dna_codes(s):
    return ["ACGT".index(c) for c in s.upper()]


def triplet_codes(s):
    d = dna_codes(s)
    return [16 * d[i] + 4 * d[i + 1] + d[i + 2] for i in range(0, len(d) - len(d) % 3, 3)]


def fold64(hi, lo):                            # A21, restated with Python integers
    t = (hi * 0x9E3779B97F4A7C15) & M64
    return lo ^ (((t << 32) | (t >> 32)) & M64)


def rand_protein(seed, n):
    r = seqgen.uniform(seed, 3 * n).astype(np.int64).reshape(n, 3)      # three uniform bases -> 64 values -> mod 26
    idx = (((r[:, 0] >> 1) & 3) * 16 + ((r[:, 1] >> 1) & 3) * 4 + ((r[:, 2] >> 1) & 3)) % 26
    return np.frombuffer(AA.encode(), dtype=np.uint8)[idx].copy()


# ---------------------------------------------------------------- W4: symbol codes
def test_w4_symbol_codes_every_byte_and_every_codon():
    for c in range(256):
        ch = bytes([c])
        want = AA.index(chr(c).upper()) if chr(c).upper() in AA and chr(c).isascii() and chr(c).isalpha() else -1
        assert oracle.symbol_code(oracle.PROTEIN, ch) == want, c
        assert oracle.symbol_code(oracle.DNA, ch) == ("ACGT".index(chr(c).upper()) if chr(c).upper() in "ACGT" else -1)
    for a in range(4):
        for b in range(4):
            for c in range(4):
                cod = ("ACGT"[a] + "acgt"[b] + "ACGT"[c]).encode()
                assert oracle.symbol_code(oracle.TRIPLET, cod) == 16 * a + 4 * b + c
    for bad in (b"ANA", b"NAA", b"AAN", b"AC-", b"\x00CG"):
        assert oracle.symbol_code(oracle.TRIPLET, bad) == -1


# ---------------------------------------------------------------- W2: big-int vectors of fold / g / f on wide windows
def _cfg_for(nbits):
    return {62: (oracle.DNA, 31), 120: (oracle.DNA, 60), 125: (oracle.PROTEIN, 25), 126: (oracle.TRIPLET, 21),
            30: (oracle.PROTEIN, 6)}[nbits]


def test_w2_wide_hash_vectors():
    n = 0
    for line in open(os.path.join(GOLD, "wide_vectors.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        lhs, rhs = line.split("=")
        name, *args = lhs.split()
        args = [int(a, 0) for a in args]
        want = int(rhs.strip(), 0)
        if name == "fold64":
            assert oracle.fold64(*args) == want, line
        else:
            nbits, hi, lo = args
            alphabet, k = _cfg_for(nbits)
            o = oracle.OracleSBF(k, k, k, 4, 1 << 16, alphabet=alphabet)     # m = s = k: ONE window, the whole k-mer
            o.force_wide(True)
            v = (hi << 64) | lo
            if name == "g_bits":
                assert o.min_key_w(v) == want, line
            else:                                                            # f: read the four bits it sets (A5)
                o.insert_kmer_w(v)
                words = o.words()
                sh = o.shard_of_w(v)
                assert [int(words[sh, i]) for i in range(4)] == [1 << ((want >> (16 * i)) & 63) for i in range(4)], line
                assert int(np.count_nonzero(words)) == 4
            o.close()
        n += 1
    assert n == 18


# ---------------------------------------------------------------- W1: DNA, k <= 32 through the wide functions == narrow path
@pytest.mark.parametrize("k,m,s,H", [(31, 16, 28, 4), (32, 16, 28, 4), (21, 11, 21, 3), (9, 5, 6, 4), (15, 15, 12, 12), (1, 1, 1, 1)])
def test_w1_wide_functions_reduce_to_the_narrow_path(k, m, s, H):
    rng = np.random.default_rng(k)
    seq = seqgen.uniform(3 + k, 30_000)
    seq[rng.integers(0, seq.size, 25)] = ord("N")
    seq[100:140] |= 0x20
    offs = np.concatenate(([0], np.sort(rng.integers(0, seq.size, 40)), [seq.size])).astype(np.uint64)
    q = seqgen.uniform(99, 20_000); q[:8000] = seq[5000:13000]
    narrow = oracle.OracleSBF(k, m, s, H, 1 << 18)
    wide = oracle.OracleSBF(k, m, s, H, 1 << 18)
    wide.force_wide(True)
    assert narrow.insert_records(seq, offs) == wide.insert_records(seq, offs) == wide.count_valid_kmers(seq, offs)
    assert np.array_equal(narrow.export_bits(), wide.export_bits())
    for threads in (False, True):
        nb, nc, nv = narrow.query_records(q, None, threads=threads)
        wb, wc, wv = wide.query_records(q, None, threads=threads)
        assert nv == wv and np.array_equal(nb, wb) and np.array_equal(nc, wc)
    wide2 = oracle.OracleSBF(k, m, s, H, 1 << 18); wide2.force_wide(True)
    wide2.insert_records(seq, offs, threads=True)                           # the OpenMP driver of the wide path
    assert np.array_equal(wide2.export_bits(), narrow.export_bits())
    # single k-mers
    for p in range(0, 300, 7):
        v = narrow.pack_kmer(seq, p)
        assert wide.pack_kmer_w(seq, p) == v
        if v is not None:
            assert wide.min_key_w(v) == narrow.min_key(v) and wide.shard_of_w(v) == narrow.shard_of(v)
            assert wide.contains_kmer_w(v) == narrow.contains_kmer(v)


# ---------------------------------------------------------------- W3: packing and sub-windows against plain strings
CASES = [(oracle.DNA, 63, 31, 60, 2), (oracle.DNA, 40, 20, 33, 2), (oracle.PROTEIN, 25, 7, 20, 5), (oracle.PROTEIN, 12, 6, 10, 5),
         (oracle.TRIPLET, 21, 9, 18, 6), (oracle.TRIPLET, 10, 5, 8, 6)]


def _random_text(alphabet, seed, n):
    return rand_protein(seed, n) if alphabet == oracle.PROTEIN else seqgen.uniform(seed, n)


def _codes(alphabet, text):
    s = text.tobytes().decode()
    return ([AA.index(c) for c in s.upper()] if alphabet == oracle.PROTEIN else
            dna_codes(s) if alphabet == oracle.DNA else triplet_codes(s))


@pytest.mark.parametrize("alphabet,k,m,s,bits", CASES)
def test_w3_pack_and_subwindows_equal_string_extraction(alphabet, k, m, s, bits):
    step = 3 if alphabet == oracle.TRIPLET else 1
    text = _random_text(alphabet, 17 + k, 400 * step)
    codes = _codes(alphabet, text)
    o = oracle.OracleSBF(k, m, s, 4, 1 << 16, alphabet=alphabet)
    for sym0 in (0, 1, 5, 77, len(codes) - k):
        v = o.pack_kmer_w(text, sym0 * step)
        assert v == pack_syms(codes[sym0:sym0 + k], bits)
        for ln in (m, s, k, 1):
            for i in sorted({0, min(1, k - ln), k - ln}):
                w = pack_syms(codes[sym0 + i:sym0 + i + ln], bits)
                assert o.sub_w(v, i, ln) == fold64(w >> 64, w & M64), (i, ln)
        # min key = minimum over the k-m+1 string-extracted m-mers of the vector-pinned g
        om = oracle.OracleSBF(m, m, m, 4, 1 << 16, alphabet=alphabet); om.force_wide(True)
        keys = [om.min_key_w(pack_syms(codes[sym0 + i:sym0 + i + m], bits)) for i in range(k - m + 1)]
        assert o.min_key_w(v) == min(keys)
    # existence: past the end, and (triplets) off the 3-byte grid of the record
    assert o.pack_kmer_w(text, (len(codes) - k + 1) * step) is None
    if alphabet == oracle.TRIPLET:
        assert o.pack_kmer_w(text, 1) is None and o.pack_kmer_w(text, 2) is None and o.pack_kmer_w(text, 3) is not None
    bad = text.copy(); bad[5 * step + step - 1] = ord("*") if alphabet == oracle.PROTEIN else ord("N")
    for sym0 in range(0, 12):
        assert (o.pack_kmer_w(bad, sym0 * step) is None) == (sym0 <= 5 < sym0 + k)


def test_w6_triplet_kmer_is_the_dna_kmer_of_three_times_the_length():
    """A codon is three bases, 6 = 3 x 2 bits, first base most significant: same packed value (A19)."""
    text = seqgen.uniform(5, 300)
    t = oracle.OracleSBF(12, 12, 12, 4, 1 << 16, alphabet=oracle.TRIPLET)
    d = oracle.OracleSBF(36, 36, 36, 4, 1 << 16, alphabet=oracle.DNA)
    for p in range(0, 150, 3):
        v = t.pack_kmer_w(text, p)
        assert v == d.pack_kmer_w(text, p) and v is not None
        assert t.min_key_w(v) == d.min_key_w(v) and t.shard_of_w(v) == d.shard_of_w(v)   # w = 1, one 72-bit window
    t.insert_records(text); d.insert_records(text)
    bt, bd = t.export_bits(), d.export_bits()
    assert np.array_equal(bt & bd, bt) and not np.array_equal(bt, bd)        # the DNA filter also holds frames 1 and 2


# ---------------------------------------------------------------- W5: P4 / P5 / P7 on the wide path
@pytest.mark.parametrize("alphabet,k,m,s,bits", CASES)
def test_w5_no_false_negatives_brute_force_set_and_shard_isolation(alphabet, k, m, s, bits):
    step = 3 if alphabet == oracle.TRIPLET else 1
    H = 4
    text = _random_text(alphabet, 41 + k, 600 * step)
    text[200 * step] = ord("*") if alphabet == oracle.PROTEIN else ord("N")
    offs = np.array([0, 250 * step + 1, 250 * step + 1, 420 * step + 2, text.size], dtype=np.uint64)   # ragged, one empty record
    o = oracle.OracleSBF(k, m, s, H, 1 << 14, alphabet=alphabet)
    n_ins = o.insert_records(text, offs)
    # brute force: the exact set of valid k-mers as strings, record by record, on each record's own symbol grid
    members, starts = set(), []
    raw = text.tobytes()
    valid_sym = (set(AA.encode()) | set(AA.lower().encode())) if alphabet == oracle.PROTEIN else set(b"ACGTacgt")
    for r in range(offs.size - 1):
        a, e = int(offs[r]), int(offs[r + 1])
        for p in range(a, e - k * step + 1, step):
            w = raw[p:p + k * step]
            if all(c in valid_sym for c in w):
                members.add(w.upper()); starts.append(p)
    assert n_ins == len(starts) > 300
    bm, counts, nv = o.query_records(text, offs)
    bits_set = oracle.bitmap_bits(bm, text.size)
    assert nv == n_ins and sorted(np.flatnonzero(bits_set)) == sorted(starts)          # P4: all true, nothing else set
    assert int(counts.sum()) == len(starts)
    # aliens: positives that are not members are false positives; members are never missed (P5)
    q = _random_text(alphabet, 1234 + k, 3000 * step)
    q[:300 * step] = text[:300 * step]
    qb, _, _ = o.query_records(q, None)
    qbits = oracle.bitmap_bits(qb, q.size)
    qraw = q.tobytes()
    for p in range(0, q.size - k * step + 1, step):
        w = qraw[p:p + k * step]
        if all(c in valid_sym for c in w) and w.upper() in members:
            assert qbits[p], p
    # P7: one k-mer changes at most H (k-s+1) bits, all inside its shard's 32 bytes
    o2 = oracle.OracleSBF(k, m, s, H, 1 << 14, alphabet=alphabet)
    v = o2.pack_kmer_w(text, 0)
    o2.insert_kmer_w(v)
    w = o2.words()
    touched = np.flatnonzero(w.any(axis=1))
    assert list(touched) == [o2.shard_of_w(v)]
    nbits = sum(bin(int(x)).count("1") for x in w[touched[0]])
    assert 1 <= nbits <= H * (k - s + 1) and o2.contains_kmer_w(v)


# ---------------------------------------------------------------- W7: minimizer density on the wide path
@pytest.mark.parametrize("alphabet,k,m,bits", [(oracle.DNA, 63, 31, 2), (oracle.PROTEIN, 12, 6, 5), (oracle.PROTEIN, 25, 13, 5),
                                               (oracle.TRIPLET, 21, 11, 6)])
def test_w7_minimizer_density(alphabet, k, m, bits):
    """Runs per k-mer = 2 / (w + 1) on random symbols, w = k - m + 1; +-6 % on 40 000 k-mers."""
    step = 3 if alphabet == oracle.TRIPLET else 1
    n = 40_000
    text = _random_text(alphabet, 7 + k, (n + k) * step)
    o = oracle.OracleSBF(k, m, k, 1, 1 << 20, alphabet=alphabet)
    keys = np.array([o.min_key_w(o.pack_kmer_w(text, p * step)) for p in range(n)], dtype=np.uint64)
    runs = 1 + int(np.count_nonzero(keys[1:] != keys[:-1]))
    w = k - m + 1
    assert abs(runs / n - 2.0 / (w + 1)) < 0.06 * 2.0 / (w + 1)


# ---------------------------------------------------------------- W8: FPR against the per-shard fill product (Eq. (1)/(2))
def _fill_product_fpr(o, H, z1):
    words = o.words()
    pc = np.zeros(words.shape, dtype=np.float64)
    for b in range(64):
        pc += ((words >> np.uint64(b)) & np.uint64(1)).astype(np.float64)
    fill = pc / 64.0
    per_shard = np.ones(words.shape[0])
    for i in range(H):
        per_shard *= fill[:, i % 4] ** z1
    return float(per_shard.mean())


@pytest.mark.parametrize("alphabet,k,m,s,H,log2_bits", [(oracle.DNA, 63, 31, 60, 4, 21), (oracle.PROTEIN, 12, 6, 10, 4, 21),
                                                        (oracle.DNA, 31, 16, 28, 12, 22)])
def test_w8_fpr_matches_the_per_shard_fill_product(alphabet, k, m, s, H, log2_bits):
    """P8 for the wide f (windows folded from 120 bits), for the protein alphabet, and — on the NARROW path — for the
    H > 10 salted bit positions (A6), which had only a big-int pin: measured FPR on uniform aliens within +-12 % (+ 3
    sigma) of the mean over shards of prod_i fill(word i mod 4)^(k-s+1)."""
    step = 3 if alphabet == oracle.TRIPLET else 1
    ins = _random_text(alphabet, 51 + k + H, 200_000 * step)
    o = oracle.OracleSBF(k, m, s, H, 1 << log2_bits, alphabet=alphabet)
    o.insert_records(ins, np.arange(0, ins.size + 1, 20_000 * step, dtype=np.uint64), threads=True)
    n_q = 400_000
    q = _random_text(alphabet, 777 + k, n_q * step)
    qoffs = np.arange(0, q.size + 1, 40_000 * step, dtype=np.uint64)
    bm, counts, nv = o.query_records(q, qoffs, threads=True)
    measured = int(counts.sum()) / nv
    predicted = _fill_product_fpr(o, H, k - s + 1)
    sigma = (predicted * (1 - predicted) / nv) ** 0.5
    assert predicted > 1e-4, "pick a smaller filter: nothing to measure"
    assert abs(measured - predicted) < 0.12 * predicted + 3 * sigma, (measured, predicted)

"""GPU parity of EVERY specialised instance of BASELINE.json config 5: all 125 (s, m, H) points at k = 31.

Each (s, m, H) is its own template instantiation (its own sliding-minimum shape, sliding-OR shape and bit-slice
layout), so "one passed" says nothing about the next: each one is compared with the oracle, bit for bit, on the slice
SURVEY.md §8(d) names — the first 5 Mbp of the config-3 sequence (it contains N runs) and its first 10^5 reads, filter
2^26 bits — through all three kernels of the instance: the insert kernel (filter bytes), the record-mode query kernel
(bitmap + per-read counts) and the chunk-mode query kernel (sbf_query_seq over a 2 Mbp stretch of the sequence: all
valid k-mers true)."""
import numpy as np
import pytest

import oracle
import seqgen
import paper_2606_24417_b200 as sbf

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

N_BASES, N_READS, NUM_BITS = 5_000_000, 100_000, 1 << 26
_cache = {}


def _inputs():
    if not _cache:
        w = seqgen.config3(scale=0.1)                     # 25 Mbp; recipe identical to config 3 (seeds 31/32/33)
        seq = np.ascontiguousarray(w.insert_bases[:N_BASES])
        w.insert_bases = seq                              # reads sampled from the slice that is inserted
        reads = w.read_batch(0, N_READS)
        offs = seqgen.fixed_offsets(N_READS, w.read_len)
        # a stretch for the chunk-mode query that contains an N run if the slice has one, else plant a short one
        sub = seq[1_000_000:3_000_000].copy()
        sub[700_000:700_050] = ord("N")
        _cache.update(seq=seq, reads=reads, offs=offs, sub=sub,
                      d_seq=torch.from_numpy(seq).cuda(), d_reads=torch.from_numpy(reads).cuda(),
                      d_offs=torch.from_numpy(offs.view(np.int64)).cuda(), d_sub=torch.from_numpy(sub).cuda())
    return _cache


@pytest.mark.parametrize("s", seqgen.SWEEP_S)
@pytest.mark.parametrize("m", seqgen.SWEEP_M)
def test_all_H_instances_of_one_s_m_pair(s, m):
    c = _inputs()
    for H in seqgen.SWEEP_H:
        params = dict(k=31, m=m, s=s, H=H)
        o = oracle.OracleSBF(num_bits=NUM_BITS, **params)
        o.insert_records(c["seq"], threads=True)
        with sbf.SuperBloomFilter(num_bits=NUM_BITS, **params) as f:
            assert f.specialized, "no specialised instance for %r" % (params,)
            f.insert_seq(c["d_seq"])
            torch.cuda.synchronize()
            got, want = f.export_bits(), o.export_bits()
            assert np.array_equal(got, want), "%r: filter differs in %d bytes" % (params, np.count_nonzero(got != want))
            bm = torch.full(((c["reads"].size + 31) // 32,), -1, dtype=torch.int32, device="cuda")
            hc = torch.full((N_READS,), -1, dtype=torch.int32, device="cuda")
            f.query_records(c["d_reads"], c["d_offs"], bm, hc)
            torch.cuda.synchronize()
            wbm, wc, _ = o.query_records(c["reads"], c["offs"], threads=True)
            assert np.array_equal(bm.cpu().numpy().view(np.uint32), wbm), "%r: record-mode bitmap differs" % (params,)
            assert np.array_equal(hc.cpu().numpy().view(np.uint32), wc), "%r: hit counts differ" % (params,)
            bm2 = torch.full(((c["sub"].size + 31) // 32,), -1, dtype=torch.int32, device="cuda")
            hits = torch.full((1,), -1, dtype=torch.int64, device="cuda")
            f.query_seq(c["d_sub"], bm2, hits)
            torch.cuda.synchronize()
            wbm2, wc2, nv = o.query_records(c["sub"], None, threads=True)
            assert np.array_equal(bm2.cpu().numpy().view(np.uint32), wbm2), "%r: chunk-mode bitmap differs" % (params,)
            assert int(hits.item()) == int(wc2.sum()) == nv       # no false negatives
        o.close()

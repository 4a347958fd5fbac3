"""bench.py's own bookkeeping (valid k-mer counts that turn times into k-mers/s) against the oracle's count."""
import numpy as np

import bench
import oracle
import seqgen


def test_valid_kmer_counts_match_the_oracle():
    w = seqgen.config3(scale=0.004)
    w.insert_bases[12345:12400] = ord("n")
    o = oracle.OracleSBF(31, 16, 28, 4, 1 << 20)
    assert bench.count_valid_kmers_seq(w.insert_bases, 31) == o.count_valid_kmers(w.insert_bases)
    reads = w.read_batch(0, 5000)
    reads[150 * 7 + 3] = ord("N")
    offs = seqgen.fixed_offsets(5000, 150)
    assert bench.count_valid_kmers_reads(reads, 150, 31) == o.count_valid_kmers(reads, offs)
    assert bench.count_valid_kmers_seq(np.frombuffer(b"ACGT" * 5, dtype=np.uint8), 31) == 0


def test_reference_arm_line_has_the_contract_keys(capsys):
    import json, sys
    argv = sys.argv
    sys.argv = ["bench.py", "--impl", "reference", "--steps", "1", "--warmup", "0", "--ref-scale", "0.004",
                "--ref-insert-bases", "200000", "--ref-reads", "500"]
    try:
        assert bench.main() == 0
    finally:
        sys.argv = argv
    line = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in line
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0


def test_sweep_helpers():
    from paper_2606_24417_b200 import sweep
    seq = np.frombuffer(b"ACGTNACGTACGTAC", dtype=np.uint8)
    assert sweep._valid_windows(seq, 4) == 1 + 7           # ACGT | ACGTACGTAC has 7 windows of 4
    reads = np.frombuffer(b"ACGTACGT" + b"ACNTACGT", dtype=np.uint8)
    assert list(sweep._valid_per_read(reads, 8, 3)) == [6, 3]
    pts = [dict(fpr_random=1e-3, time_ms=2.0), dict(fpr_random=1e-4, time_ms=3.0), dict(fpr_random=1e-3, time_ms=2.5),
           dict(fpr_random=1e-5, time_ms=3.0)]
    assert sweep.pareto(pts) == [0, 3]                     # 2 is dominated by 0, 1 by 3

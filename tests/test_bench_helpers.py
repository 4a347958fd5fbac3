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

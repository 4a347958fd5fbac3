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


def test_instruction_roofline_model():
    """alu_roofline: the peak is the measured issue rate of the ALGORITHMIC alu:fma mix; executed counts give busy fractions."""
    ceil = {"pipe_warp_inst_per_clk_per_smsp": {"LOP3": 0.5, "IMAD": 0.5, "LOP3:IMAD 1:1": 1.0}}
    ops = {"alu": 56.0, "fma": 7.0}
    # 592 SMSPs at 1000 MHz; the alu pipe binds: 56 / 0.5 = 112 clocks per warp of 32 k-mers
    n, ms = 32 * 592 * 1000, 1.0
    r = bench.alu_roofline(ops, n, ms, ceil, 1000.0, None)
    ideal_ms = 112 * 1000 / 1000e6 * 1e3
    assert abs(r["frac"] - ideal_ms / ms) < 1e-9 and r["bound"] == "alu"
    assert abs(r["peak"] - 63.0 / 112.0 * 32 * 592 * 1e9 / 1e12) < 1e-9
    ex = {"units": float(n), "inst_total": 90.0 * n / 32, "inst_alu": 57.0 * n / 32, "inst_fma": 16.0 * n / 32}
    r = bench.alu_roofline(ops, n, ms, ceil, 1000.0, ex)
    cyc = 1e-3 * 1000e6 * 592
    assert abs(r["busy_fraction_of_measured_limit"]["alu_pipe"] - (57.0 * n / 32) / 0.5 / cyc) < 1e-9
    assert r["binding_instruction_limit"] == "alu_pipe"
    assert abs(r["executed_warp_inst_per_kmer"]["alu"] - 57.0) < 1e-9
    # an fma-heavy mix is bound by issue, not by either pipe
    r = bench.alu_roofline({"alu": 30.0, "fma": 30.0}, n, ms, ceil, 1000.0, None)
    assert abs(r["peak"] - 1.0 * 32 * 592 * 1e9 / 1e12) < 1e-9
    # wide multiplies (IMAD.WIDE / IMAD.HI) add their measured cost to the alu-pipe time: LOP3:IMAD.HI 3:1 at 4/9 per clock
    # means 3 LOP3 (6 clocks) + 1 IMAD.HI take 9 clocks, i.e. 3 clocks per wide multiply
    ceil["pipe_warp_inst_per_clk_per_smsp"]["LOP3:IMAD.HI 3:1"] = 4.0 / 9.0
    r = bench.alu_roofline({"alu": 40.0, "fma": 4.0, "wide": 4.0}, n, ms, ceil, 1000.0, None, survey_ops=63.0)
    assert abs(r["peak"] - 48.0 / (80.0 + 12.0) * 32 * 592 * 1e9 / 1e12) < 1e-6
    assert abs(r["frac_with_survey_count"] - 63.0 * n / 1e-3 / (32 * 592 * 1e9 * 0.5)) < 1e-9


def test_static_profile_tables_load():
    rows = bench.load_csv_rows("profiles/traffic.csv")
    assert rows and {"kernel", "dram_bytes_per_launch", "source"} <= set(rows[0])
    t, src = bench.load_traffic("query_kernel")
    assert t > 0 and "ncu" in src

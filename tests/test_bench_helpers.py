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


def _kernel_entry(frac_alu, frac_rs, frac_hbm, ms):
    return {"achieved": 10.0 * frac_alu, "peak": 10.0, "frac": frac_alu, "frac_with_survey_count": frac_alu * 1.4, "ms": ms,
            "algorithmic_ops_per_kmer": {"alu": 39.0, "fma": 4.0, "wide": 3.0}, "survey_planning_ops_per_kmer": 63.0,
            "peak_source": "x", "binds": max((("alu_pipe", frac_alu), ("random_sector", frac_rs), ("hbm_bytes", frac_hbm)),
                                              key=lambda kv: kv[1])[0],
            "binds_busy": max(frac_alu, frac_rs, frac_hbm),
            "random_sector": {"achieved_g_per_s": 48.0 * frac_rs, "ceiling_g_per_s": 48.0, "frac": frac_rs, "ceiling": "loads"},
            "hbm": {"achieved": 6000.0 * frac_hbm, "peak": 6000.0, "unit": "GB/s", "frac": frac_hbm, "peak_source": "m"}}


def test_top_roofline_quotes_the_binding_limit():
    """roofline.bound / frac follow the limit that binds; the instruction fractions (both counts) stay beside it."""
    r = bench.top_roofline(_kernel_entry(0.80, 0.92, 0.30, 1.5), "query_kernel", 123, "src")
    assert r["bound"] == "hbm" and r["binds"] == "random_sector" and r["unit"] == "GB/s"
    assert abs(r["frac"] - 0.92) < 1e-12 and abs(r["achieved"] / r["peak"] - r["frac"]) < 1e-12
    assert r["alu"]["frac"] == 0.80 and r["alu"]["ops_per_kmer"] == 46.0 and r["alu"]["survey_ops_per_kmer"] == 63.0
    assert r["traffic"] == 123 and r["kernel"] == "query_kernel"
    r = bench.top_roofline(_kernel_entry(0.85, 0.50, 0.30, 1.5), "query_kernel", None, None)
    assert r["bound"] == "alu" and r["frac"] == 0.85 and r["unit"] == "Tiop/s"
    r = bench.top_roofline(_kernel_entry(0.2, 0.3, 0.7, 1.5), "insert_kernel", None, None)
    assert r["bound"] == "hbm" and r["limit"] == "streamed bytes" and r["frac"] == 0.7


def test_step_roofline_adds_up():
    roof = {"insert_kernel": _kernel_entry(0.7, 0.97, 0.3, 1.2), "query_kernel": _kernel_entry(0.8, 0.9, 0.3, 1.4)}
    s = bench.step_roofline(roof, 2.9, pack_bytes=6.0e8, clear_bytes=4.0e8, hbm_gbs=5000.0)
    want = 1.2 * 0.97 + 1.4 * 0.9 + 1.0e9 / 5.0e12 * 1e3
    assert abs(s["roofline_ms"] - want) < 1e-9 and abs(s["frac"] - want / 2.9) < 1e-9
    assert abs(sum(s["parts_ms"].values()) - s["roofline_ms"]) < 1e-9

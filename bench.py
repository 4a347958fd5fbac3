#!/usr/bin/env python
"""bench.py — throughput of the Super Bloom filter insert + query hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload config3]

One STEP = one pass of the whole hot path over one batch of the
workload: clear the filter, insert the workload's sequence (pack -> fused minimizer / shard /
s-mer / merge kernel), [N>1: OR all-reduce of the replicas], query one batch of reads (pack ->
fused query kernel -> packed bitmap -> per-record hit counts).  `value` = valid k-mers inserted
+ valid k-mers queried by all ranks, per second of device time (max over ranks).

Default workload: BASELINE.json configs[2] (the out-of-L2 config north_star's target is quoted
on): 250 Mbp order-5 Markov sequence with N runs, k=31 m=16 s=28 H=4, filter 2^32 bits; reads of
length 150 (half sampled with 1% substitutions, half uniform), queried in batches.  All inputs are
seeded synthetic stand-ins (seqgen/), see DESIGN.md "Input recipe".

The product path is the C ABI (include/sbf.h) through its ctypes binding; the oracle is executed
only by the `cpu_baseline` leg and by `--impl reference`.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "G k-mers/s insert+query (1 step = insert the sequence + query one read batch)"
# ALGORITHMIC integer instructions per valid k-mer of the fused kernels (defaults k=31 m=16 s=28 H=4), derived part by part in
# DESIGN.md §6, split by how they issue: "alu" (LOP3/SHF/PRMT/VIMNMX/ISETP class), "fma" (32-bit IMAD / IDP.4A: the
# fma pipe at full rate), "wide" (IMAD.WIDE / IMAD.HI, the 64-bit-result multiplies of sigma, f and the sector
# address: half rate and, measured, not overlapping the alu pipe).  SURVEY.md §8(d)'s planning figures
# were 70 (insert) and 63 (query); the query's byte-gather formulation of round 2 needs fewer (the survey's 26 for the bit
# tests became 21), so it is restated here — quoting the kernel against the survey's 63 would give a fraction above 1.
OPS_PER_KMER = {"insert": {"alu": 63.0, "fma": 5.0, "wide": 2.0}, "query": {"alu": 39.0, "fma": 4.0, "wide": 3.0}}
SURVEY_OPS_PER_KMER = {"insert": 70.0, "query": 63.0}
N_SMSP = 148 * 4
# What the kernels EXECUTE (warp instructions per launch, by pipe): ncu counters of a committed capture, static.
PIPES_CSV = os.path.join("profiles", "pipes_r02.csv")


def env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            d = json.load(fh)
        return float(d.get("hbm_gbs", 6650.0)), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


# ------------------------------------------------------------------------------------------------
# workload
# ------------------------------------------------------------------------------------------------
def make_workload(name: str, rank: int, scale: float):
    import seqgen
    if name == "config3":
        w = seqgen.config3(scale=scale)
    elif name == "config2":
        w = seqgen.config2(scale=scale)
        w.params["num_bits"] = 1 << 27
    elif name == "config1":
        w = seqgen.config1()
        w.n_reads = 6000
        w.read_seed = 3
    elif name == "config4":
        w = seqgen.config4(scale=scale)
    else:
        raise SystemExit("unknown workload %r" % name)
    if rank:  # weak scaling: every rank owns an independent sequence of the same recipe
        n = w.insert_bases.size
        if name == "config3":
            seq = seqgen.markov(31 + 1000 * rank, 5, 0.41, n)
            seqgen.plant_n_runs(32 + 1000 * rank, seq, max(1, int(round(100 * scale))), 10_000, 50_000)
        elif name == "config2":
            seq = seqgen.markov(21 + 1000 * rank, 3, 0.50, n)
            seqgen.plant_copies(22 + 1000 * rank, seq, max(1, int(200 * scale)), 1000, 5000, 0.005)
        elif name == "config4":
            seq = seqgen.markov(41 + 1000 * rank, 5, 0.41, n)
            seqgen.plant_families(42 + 1000 * rank, seq, [300] * 6 + [6000] * 2, 0.05, 0.10, 0.20)
        else:
            seq = seqgen.uniform(1 + 1000 * rank, n)
        w.insert_bases = seq
        w.read_seed += 1000 * rank
    return w


_ACGT = np.zeros(256, dtype=bool)
for _c in b"ACGTacgt":
    _ACGT[_c] = True


def count_valid_kmers_seq(seq: np.ndarray, k: int) -> int:
    """k-mer windows of one sequence without a non-ACGT symbol (harness bookkeeping for the metric)."""
    n = seq.size
    if n < k:
        return 0
    total, step = 0, 1 << 26
    for a in range(0, n - k + 1, step):
        e = min(a + step + k - 1, n)
        bad = ~_ACGT[seq[a:e]]
        if not bad.any():
            total += e - a - k + 1
            continue
        cs = np.concatenate(([0], np.cumsum(bad, dtype=np.int32)))
        total += int(np.count_nonzero(cs[k:] - cs[:-k] == 0))
    return total


def count_valid_kmers_reads(reads: np.ndarray, read_len: int, k: int) -> int:
    n = reads.size // read_len
    per = max(read_len - k + 1, 0)
    bad_rows = np.flatnonzero((~_ACGT[reads]).reshape(n, read_len).any(axis=1))
    total = (n - bad_rows.size) * per
    for r in bad_rows:
        total += count_valid_kmers_seq(reads[r * read_len:(r + 1) * read_len], k)
    return total


# ------------------------------------------------------------------------------------------------
# clocks
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS, "--format=csv,noheader,nounits",
                 "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append((time.perf_counter(), ln.strip()))

    def stop(self, t0: float, t1: float):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for t, ln in self.lines:
            if t < t0 or t > t1 + 0.06:
                continue
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); pw.append(float(parts[2]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:  # region shorter than the sampling period: take whatever was seen
            for t, ln in self.lines[-3:]:
                parts = [x.strip() for x in ln.split(",")]
                try:
                    sm.append(float(parts[0])); mx.append(float(parts[1])); pw.append(float(parts[2]))
                except (ValueError, IndexError):
                    pass
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
# the oracle on the host cores (cpu_baseline leg and --impl reference): bounded sample
# ------------------------------------------------------------------------------------------------
def oracle_sample_step(o, seq_sample, reads_sample, offs_sample, threads: bool):
    """One oracle 'step' on the bounded sample: clear, insert, query.  Returns (k-mers, seconds)."""
    o.clear()                                   # the 512 MiB memset is not part of the oracle's insert rate
    t0 = time.perf_counter()
    n_ins = o.insert_records(seq_sample, threads=threads)
    t1 = time.perf_counter()
    _, counts, n_q = o.query_records(reads_sample, offs_sample, want_counts=True, threads=threads)
    t2 = time.perf_counter()
    oracle_sample_step.last_counts = counts
    return n_ins, n_q, t1 - t0, t2 - t1


def make_oracle_sample(w, ins_bases: int, n_reads: int):
    import seqgen
    seq_sample = np.ascontiguousarray(w.insert_bases[:ins_bases])
    reads_sample = w.read_batch(0, n_reads)
    offs = seqgen.fixed_offsets(n_reads, w.read_len)
    return seq_sample, reads_sample, offs


def run_reference(args):
    """--impl reference: the oracle as it stands, all host cores (its OpenMP driver), bounded sample."""
    rank = env_int("RANK", 0)
    if rank != 0:
        return 0
    import oracle
    w = make_workload(args.workload, 0, args.ref_scale)
    p = w.params
    ins_bases = min(w.insert_bases.size, args.ref_insert_bases)
    n_reads = min(max(w.n_reads, 1), args.ref_reads)
    seq_s, reads_s, offs_s = make_oracle_sample(w, ins_bases, n_reads)
    o = oracle.OracleSBF(p["k"], p["m"], p["s"], p["H"], p["num_bits"])
    cores = oracle.num_threads()
    for _ in range(args.warmup):
        oracle_sample_step(o, seq_s, reads_s, offs_s, True)
    kmers, secs, ti, tq, ni, nq = 0, 0.0, 0.0, 0.0, 0, 0
    for _ in range(args.steps):
        a, b, t_i, t_q = oracle_sample_step(o, seq_s, reads_s, offs_s, True)
        kmers += a + b; secs += t_i + t_q; ti += t_i; tq += t_q; ni += a; nq += b
    val = kmers / secs / 1e9
    sample = "per step: insert first %d bases of the %s sequence + query first %d reads x %d" % (
        ins_bases, args.workload, n_reads, w.read_len)
    line = {
        "impl": "reference", "metric": METRIC, "value": val,
        "unit": "G k-mers/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": secs / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u64", "data": "synthetic",
        "config": {"workload": args.workload, "k": p["k"], "m": p["m"], "s": p["s"], "H": p["H"],
                   "filter_bits": o.num_bits, "sample": sample},
        "insert_gkmers_s": ni / ti / 1e9, "query_gkmers_s": nq / tq / 1e9,
        "cpu_baseline": {"value": val, "unit": "G k-mers/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "G k-mers/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------
def run_cuda(args):
    import torch
    import torch.distributed as dist
    import seqgen
    import paper_2606_24417_b200 as sbf
    from paper_2606_24417_b200 import replicas

    world = env_int("WORLD_SIZE", 1)
    rank = env_int("RANK", 0)
    local_rank = env_int("LOCAL_RANK", 0)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — this framework has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    sbf.load_library(build_if_missing=True)
    hbm_gbs, sm_max_mhz, peak_src = load_peaks()

    # ---- inputs (host, pinned) -> device -------------------------------------------------------
    w = make_workload(args.workload, rank, args.scale)
    p = w.params
    k = p["k"]
    seq_h = torch.from_numpy(w.insert_bases).pin_memory()
    ins_offs_np = np.ascontiguousarray(w.insert_offsets, dtype=np.uint64)
    n_ins_rec = ins_offs_np.size - 1
    n_ins_kmers = sum(count_valid_kmers_seq(w.insert_bases[int(ins_offs_np[r]):int(ins_offs_np[r + 1])], k)
                      for r in range(n_ins_rec))
    rb = min(args.read_batch, max(w.n_reads, 1))
    n_batches = max(1, min(args.batches, max(w.n_reads, 1) // rb))
    offs_np = seqgen.fixed_offsets(rb, w.read_len)
    reads_h, n_q_kmers = [], []
    for b in range(n_batches):
        t = torch.empty(rb * w.read_len, dtype=torch.uint8).pin_memory()
        w.read_batch(b * rb, rb, out=t.numpy())
        reads_h.append(t)
        n_q_kmers.append(count_valid_kmers_reads(t.numpy(), w.read_len, k))
    offs_h = torch.from_numpy(offs_np.view(np.int64)).pin_memory()

    d_seq = seq_h.cuda(non_blocking=True)
    d_ins_offs = torch.from_numpy(ins_offs_np.view(np.int64)).cuda()

    def do_insert(st):  # one sequence, or a dense record batch (config 4)
        if n_ins_rec == 1:
            sbf.sbf_insert_seq(h, d_seq, d_seq.numel(), st)
        else:
            sbf.sbf_insert_records(h, d_seq, d_ins_offs, n_ins_rec, d_seq.numel(), st)
    d_reads = [t.cuda(non_blocking=True) for t in reads_h]
    d_offs = offs_h.cuda(non_blocking=True)
    n_read_bases = rb * w.read_len
    d_bitmap = torch.empty((n_read_bases + 31) // 32, dtype=torch.int32, device="cuda")
    d_counts = torch.empty(rb, dtype=torch.int32, device="cuda")
    h_bitmap = torch.empty((n_read_bases + 31) // 32, dtype=torch.int32).pin_memory()
    h_counts = torch.empty(rb, dtype=torch.int32).pin_memory()
    torch.cuda.synchronize()

    h = sbf.sbf_create(k, p["m"], p["s"], p["H"], p["num_bits"])
    num_bits = sbf.sbf_num_bits(h)
    sbf.sbf_reserve(h, max(d_seq.numel(), n_read_bases))
    sbf.sbf_set_timing(h, True)
    stream = torch.cuda.current_stream()

    def step(i: int, ev=None):
        b = i % n_batches
        if ev: ev[0].record(stream)
        sbf.sbf_clear(h, stream)
        do_insert(stream)
        if world > 1:
            replicas.or_allreduce_filter(h, stream=stream)
        if ev: ev[1].record(stream)
        sbf.sbf_query_records(h, d_reads[b], d_offs, rb, n_read_bases, d_bitmap, d_counts, stream)
        if ev: ev[2].record(stream)
        return b

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- warm-up, then the timed region ----------------------------------------------------------
    for i in range(args.warmup):
        step(i)
    barrier()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    ins_kernel_ms, q_kernel_ms, pack_ms, count_ms = [], [], [], []
    sampler = ClockSampler(local_rank if "CUDA_VISIBLE_DEVICES" not in os.environ else
                           int(os.environ["CUDA_VISIBLE_DEVICES"].split(",")[local_rank]))
    sampler.start()
    time.sleep(0.12)
    launches0 = sbf.sbf_kernel_launches()
    barrier()
    t_host0 = time.perf_counter()
    e_begin = torch.cuda.Event(enable_timing=True); e_end = torch.cuda.Event(enable_timing=True)
    e_begin.record(stream)
    q_total = 0
    for i in range(args.steps):
        b = step(args.warmup + i, evs[i])
        q_total += n_q_kmers[b]
    e_end.record(stream)
    barrier()
    t_host1 = time.perf_counter()
    launches = sbf.sbf_kernel_launches() - launches0
    clocks = sampler.stop(t_host0, t_host1)
    total_ms = e_begin.elapsed_time(e_end)
    ins_ms = sum(e[0].elapsed_time(e[1]) for e in evs)
    qry_ms = sum(e[1].elapsed_time(e[2]) for e in evs)

    # per-kernel device times (events the library records on the same stream around each kernel):
    # a few extra steps, same inputs, so that the two calls of a step can be read separately
    for i in range(min(args.steps, 5)):
        b = (args.warmup + i) % n_batches
        sbf.sbf_clear(h, stream)
        do_insert(stream)
        pk, mn, _ = sbf.sbf_get_timing(h)
        ins_kernel_ms.append(mn); pack_ms.append(pk)
        sbf.sbf_query_records(h, d_reads[b], d_offs, rb, n_read_bases, d_bitmap, d_counts, stream)
        pk, mn, ct = sbf.sbf_get_timing(h)
        q_kernel_ms.append((mn, n_q_kmers[b])); pack_ms.append(pk); count_ms.append(ct)
    torch.cuda.synchronize()

    ceilings = measure_ceilings(sbf, num_bits // 8, sampler.index, sm_max_mhz) if rank == 0 else None

    # measured statistics of the last query batch: FPR on the uniform reads (odd read index)
    cnt = d_counts.cpu().numpy().view(np.uint32).astype(np.int64)
    per_read = max(w.read_len - k + 1, 1)
    fpr_random = float(cnt[1::2].sum()) / max(1, cnt[1::2].size * per_read)
    hit_sampled = float(cnt[0::2].sum()) / max(1, cnt[0::2].size * per_read)

    # ---- end to end through the host-facing C ABI (pinned host buffers, H2D + D2H inside) -----------
    sbf.sbf_set_timing(h, False)
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    hb_np, hc_np = h_bitmap.numpy().view(np.uint32), h_counts.numpy().view(np.uint32)
    offs_pinned_np = offs_h.numpy().view(np.uint64)  # offsets, like every other host buffer of this leg, are pinned

    def e2e_step(i):
        b = i % n_batches
        sbf.sbf_clear(h, None)
        if n_ins_rec == 1:
            sbf.sbf_insert_seq_host(h, seq_h, seq_h.numel())
        else:
            sbf.sbf_insert_records_host(h, seq_h, ins_offs_np, n_ins_rec)
        if world > 1:
            replicas.or_allreduce_filter(h, stream=stream)
            torch.cuda.synchronize()
        sbf.sbf_query_records_host(h, reads_h[b], offs_pinned_np, rb, hb_np, hc_np)
        return b

    e2e_step(0)
    barrier()
    t0 = time.perf_counter()
    e2e_kmers = 0
    for i in range(e2e_steps):
        b = e2e_step(i + 1)
        e2e_kmers += n_ins_kmers + n_q_kmers[b]
    barrier()
    e2e_s = time.perf_counter() - t0
    h2d = seq_h.numel() + n_read_bases + offs_np.nbytes
    d2h = hb_np.nbytes + hc_np.nbytes
    # the host-facing calls must have produced what the device-facing calls produce on the same batch
    e2e_filter = sbf.sbf_export_bits(h) if world == 1 else None
    sbf.sbf_clear(h, stream)
    do_insert(stream)
    if world > 1:
        replicas.or_allreduce_filter(h, stream=stream)
    sbf.sbf_query_records(h, d_reads[b], d_offs, rb, n_read_bases, d_bitmap, d_counts, stream)
    torch.cuda.synchronize()
    e2e_ok = bool(np.array_equal(d_bitmap.cpu().numpy().view(np.uint32), hb_np)
                  and np.array_equal(d_counts.cpu().numpy().view(np.uint32), hc_np)
                  and (e2e_filter is None or np.array_equal(sbf.sbf_export_bits(h), e2e_filter)))
    del e2e_filter
    if not e2e_ok:
        raise SystemExit("bench.py: the host-facing calls and the device-facing calls disagree on the same batch")

    # ---- reduce over ranks ------------------------------------------------------------------------
    kmers_local = args.steps * n_ins_kmers + q_total
    vals = torch.tensor([total_ms, ins_ms, qry_ms, e2e_s, float(kmers_local), float(e2e_kmers),
                         float(args.steps * n_ins_kmers), float(q_total)], dtype=torch.float64, device="cuda")
    if world > 1:
        mx = vals.clone(); dist.all_reduce(mx, op=dist.ReduceOp.MAX)
        sm = vals.clone(); dist.all_reduce(sm, op=dist.ReduceOp.SUM)
        total_ms, ins_ms, qry_ms, e2e_s = (float(x) for x in mx[:4])
        kmers_all, e2e_kmers_all, ins_all, q_all = (float(x) for x in sm[4:])
    else:
        kmers_all, e2e_kmers_all, ins_all, q_all = float(kmers_local), float(e2e_kmers), float(
            args.steps * n_ins_kmers), float(q_total)

    if rank == 0:
        value = kmers_all / (total_ms * 1e-3) / 1e9
        ins_rate = ins_all / (ins_ms * 1e-3) / 1e9
        q_rate = q_all / (qry_ms * 1e-3) / 1e9
        # ---- rooflines, against ceilings measured in this run ---------------------------------
        ik = statistics.mean(ins_kernel_ms)
        qk = statistics.mean(m for m, _ in q_kernel_ms)
        qk_kmers = statistics.mean(n for _, n in q_kernel_ms)
        w_ = k - p["m"] + 1
        d_runs = 2.0 / (w_ + 1)                      # runs per k-mer on random sequence
        clock_mhz = sm_max_mhz                       # rooflines are quoted at the maximum SM clock
        ex_i, ex_i_src = load_pipes("insert_kernel")
        ex_q, ex_q_src = load_pipes("query_kernel")
        roof = {"insert_kernel": alu_roofline(OPS_PER_KMER["insert"], n_ins_kmers, ik, ceilings, clock_mhz, ex_i,
                                              SURVEY_OPS_PER_KMER["insert"]),
                "query_kernel": alu_roofline(OPS_PER_KMER["query"], qk_kmers, qk, ceilings, clock_mhz, ex_q,
                                             SURVEY_OPS_PER_KMER["query"]),
                "pack_kernel_ms_mean": statistics.mean(pack_ms), "count_kernel_ms_mean": statistics.mean(count_ms)}
        roof["insert_kernel"]["executed_source"], roof["query_kernel"]["executed_source"] = ex_i_src, ex_q_src
        # HBM: algorithmic bytes of the fused kernels (packed 2-bit words + mask + one sector read/write per run)
        ins_bytes = d_seq.numel() * (0.25 + 0.125) + n_ins_kmers * d_runs * 64.0
        q_bytes = n_read_bases * (0.25 + 0.125 + 0.125) + qk_kmers * (d_runs + 1.0 / per_read) * 32.0
        for kk, nbytes, ms_ in (("insert_kernel", ins_bytes, ik), ("query_kernel", q_bytes, qk)):
            roof[kk]["hbm"] = {"achieved": nbytes / (ms_ * 1e-3) / 1e9, "peak": hbm_gbs, "unit": "GB/s",
                               "frac": nbytes / (ms_ * 1e-3) / 1e9 / hbm_gbs,
                               "peak_source": peak_src + " (MEASURED_PEAKS.json hbm_gbs)"}
            if clocks.get("sm_mhz"):
                roof[kk]["frac_at_achieved_clock"] = roof[kk]["frac"] * clock_mhz / clocks["sm_mhz"]
        # random 32-byte-sector accesses against the ceilings measured above for exactly that access: one
        # read-modify-write (4 x RED.OR.B64) per insert run, one staged 2 x 16-byte cp.async per query run;
        # runs = k-mers x 2/(w+1) (+ one per record for the reads)
        rs = ceilings["random_sector_g_per_s"]
        ins_runs_g = n_ins_kmers * d_runs / (ik * 1e-3) / 1e9
        q_runs_g = qk_kmers * (d_runs + 1.0 / per_read) / (qk * 1e-3) / 1e9
        # the best any read-modify-write form reached (1 RED, 4 REDs, one 32-byte TMA reduction) / any load form
        rmw_ceiling = max(x for x in (rs.get("red_or_b64_x4"), rs.get("red_or_b64_x1"), rs.get("tma_reduce_or_32B")) if x)
        ld_ceiling = max(x for x in (rs.get("ld_nc_256"), rs.get("cp_async_2x16"), rs.get("ld_nc_256_L2_64B"),
                                     rs.get("cp_async_2x16_L2_64B")) if x)
        roof["insert_kernel"]["random_sector"] = {
            "achieved_g_per_s": ins_runs_g, "ceiling_g_per_s": rmw_ceiling, "frac": ins_runs_g / rmw_ceiling,
            "ceiling": "random read-modify-write sectors/s over %d MiB, best of 1 RED, 4 REDs, one TMA reduction" % (num_bits >> 23)}
        roof["query_kernel"]["random_sector"] = {
            "achieved_g_per_s": q_runs_g, "ceiling_g_per_s": ld_ceiling, "frac": q_runs_g / ld_ceiling,
            "ceiling": "random sector loads/s over %d MiB, best of one 256-bit ld.global.nc and 2 x 16-byte cp.async, "
                       "each with and without the .L2::64B hint" % (num_bits >> 23)}
        for kk in ("insert_kernel", "query_kernel"):  # which limit binds this kernel: instructions or random sectors
            r = roof[kk]
            busy = dict(r.get("busy_fraction_of_measured_limit", {"alu_pipe": r["frac"]}))
            busy["random_sector"] = r["random_sector"]["frac"]
            busy["hbm_bytes"] = r["hbm"]["frac"]
            r["binds"] = max(busy, key=busy.get)
            r["binds_busy"] = busy[r["binds"]]
        dom = "query_kernel" if qk * 1.0 >= ik else "insert_kernel"
        traffic, traffic_src = load_traffic(dom)
        roofline = top_roofline(roof[dom], dom, traffic, traffic_src)
        # the one driver-timed number against a roofline of its own: both fused kernels at the limit that binds them
        # plus the streamed bytes of the passes around them (pack: 1 B/base in, 0.375 B/base out, + the result bitmap
        # zeroed in passing for the reads; clear: the filter written once) at the measured HBM rate
        roofline["step"] = step_roofline(roof, total_ms / args.steps,
                                         pack_bytes=d_seq.numel() * 1.375 + n_read_bases * 1.5,
                                         clear_bytes=num_bits / 8.0, hbm_gbs=hbm_gbs)
        line = {
            "metric": METRIC,
            "value": value, "unit": "G k-mers/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u64", "data": "synthetic",
            "config": {"workload": args.workload, "k": k, "m": p["m"], "s": p["s"], "H": p["H"],
                       "filter_bits": num_bits, "insert_bases_per_rank": int(d_seq.numel()),
                       "insert_kmers_per_rank": int(n_ins_kmers), "insert_records": int(n_ins_rec), "reads_per_batch": rb, "read_len": w.read_len,
                       "read_batches": n_batches, "l2": "inputs larger than L2 (sequence %d MB, read batch %d MB, "
                       "filter %d MiB); no flush" % (d_seq.numel() // 10**6, n_read_bases // 10**6, num_bits >> 23),
                       "parallelism": "replicas x%d + OR all-reduce" % world if world > 1 else "single GPU"},
            "insert_gkmers_s": ins_rate, "query_gkmers_s": q_rate,
            "fpr": {"random_reads": fpr_random, "sampled_reads_hit_rate": hit_sampled,
                    "bits_per_inserted_kmer": num_bits / max(1, n_ins_kmers)},
            "clocks": clocks,
            "e2e": {"value": e2e_kmers_all / e2e_s / 1e9, "unit": "G k-mers/s", "h2d_bytes_per_step": int(h2d),
                    "d2h_bytes_per_step": int(d2h), "steps": e2e_steps,
                    "api": "sbf_insert_seq_host + sbf_query_records_host (pinned host buffers)",
                    "verified": "filter bytes, bitmap and hit counts equal the device-facing calls' on the same batch"},
            "gpu_launches": int(launches),
            "roofline": roofline, "rooflines": roof, "ceilings": ceilings,
        }
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"], sample, o_counts = cpu_baseline(args, w)
            # the same bounded sample through the CUDA path: the two FPRs are one statistic (equal by parity)
            seq_s, reads_s, offs_s = sample
            h2 = sbf.sbf_create(k, p["m"], p["s"], p["H"], p["num_bits"])
            sbf.sbf_insert_seq(h2, torch.from_numpy(seq_s).cuda(), seq_s.size)
            bm2 = torch.empty((reads_s.size + 31) // 32, dtype=torch.int32, device="cuda")
            hc2 = torch.empty(offs_s.size - 1, dtype=torch.int32, device="cuda")
            sbf.sbf_query_records(h2, torch.from_numpy(reads_s).cuda(), torch.from_numpy(offs_s.view(np.int64)).cuda(),
                                  offs_s.size - 1, reads_s.size, bm2, hc2)
            torch.cuda.synchronize()
            g_counts = hc2.cpu().numpy().view(np.uint32)
            sbf.sbf_destroy(h2)
            n_alien = max(1, g_counts[1::2].size * per_read)
            line["fpr"]["same_sample"] = {
                "sample": line["cpu_baseline"]["sample"], "gpu": float(g_counts[1::2].astype(np.int64).sum()) / n_alien,
                "oracle": float(o_counts[1::2].astype(np.int64).sum()) / n_alien,
                "hit_counts_identical": bool(np.array_equal(g_counts, o_counts))}
        print(json.dumps(line))
    sbf.sbf_destroy(h)
    if world > 1:
        dist.destroy_process_group()
    return 0


def load_csv_rows(rel):
    try:
        with open(os.path.join(ROOT, rel)) as fh:
            lines = [ln for ln in fh.read().splitlines() if ln and not ln.startswith("#")]
        hdr = lines[0].split(",")
        return [dict(zip(hdr, ln.split(","))) for ln in lines[1:]]
    except Exception:
        return []


def load_traffic(kernel: str):
    """DRAM bytes per launch of the dominant kernel (dram__bytes_read.sum + dram__bytes_write.sum of a committed
    `ncu --set full` capture, profiles/traffic.csv).  STATIC: it describes the build that was profiled, which the
    `source` column names; None until a capture exists."""
    for r in load_csv_rows(os.path.join("profiles", "traffic.csv")):
        if r.get("kernel") == kernel:
            return int(r["dram_bytes_per_launch"]), r.get("source", "profiles/traffic.csv")
    return None, None


def load_pipes(kernel: str):
    """Executed warp instructions per launch by pipe (ncu smsp__inst_executed_pipe_*.sum; static, see PIPES_CSV)."""
    for r in load_csv_rows(PIPES_CSV):
        if r.get("kernel") == kernel:
            return {k: float(v) for k, v in r.items() if k not in ("kernel", "source")}, r.get("source", PIPES_CSV)
    return None, None


class NvmlClock:
    """SM clock of one GPU sampled through NVML every few milliseconds while a block of code runs."""

    def __init__(self, index: int):
        self.h = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
        except Exception:
            self.h = None

    def during(self, fn):
        """Run fn(); return (its result, median SM clock in MHz sampled meanwhile or None)."""
        if self.h is None:
            return fn(), None
        samples, stop = [], threading.Event()

        def loop():
            while not stop.is_set():
                try:
                    samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                except Exception:
                    pass
                time.sleep(0.004)
        t = threading.Thread(target=loop, daemon=True)
        t.start()
        try:
            out = fn()
        finally:
            stop.set()
            t.join()
        tail = samples[len(samples) // 3:]          # the first third may still see the idle clock
        return out, (statistics.median(tail) if tail else None)


def measure_ceilings(sbf, filter_bytes, gpu_index, sm_max_mhz):
    """The box's ceilings, measured in THIS run through the library's sbf_ceiling_* entry points: issue rates of
    one SM sub-partition by instruction mix (warp instructions per second, counted in SASS, divided by the SM clock
    NVML reports during that very run) and random 32-byte-sector access rates over an array as large as the filter."""
    nv = NvmlClock(gpu_index)
    per_s, per_clk, clocks = {}, {}, {}
    for mode in range(sbf.sbf_ceiling_pipe_modes()):
        name = sbf.sbf_ceiling_pipe_mode_name(mode)
        (g_per_s, _c64), mhz = nv.during(lambda: sbf.sbf_ceiling_pipe_rate(mode, 24000))
        per_s[name] = g_per_s
        clocks[name] = mhz
        per_clk[name] = g_per_s * 1e3 / (mhz if mhz else sm_max_mhz)
    names = ["red_or_b64_x4", "red_or_b64_x1", "ld_nc_256", "cp_async_2x16", "tma_reduce_or_32B", "ld_nc_256_L2_64B",
             "cp_async_2x16_L2_64B", "st_256"]
    rnd = {}
    for mode, nm in enumerate(names):
        try:
            rnd[nm] = sbf.sbf_ceiling_random_sector(mode, min(filter_bytes, 8 << 30))
        except Exception:  # noqa: BLE001 - a ceiling that cannot be measured is reported as such
            rnd[nm] = None
    return {"source": "measured in this run (sbf_ceiling_pipe_rate / sbf_ceiling_random_sector, include/sbf_bench.h, libsbf_bench_b200.so)",
            "pipe_g_warp_inst_per_s_per_smsp": per_s, "sm_clock_mhz_during_pipe_runs": clocks,
            "sm_clock_source": "NVML nvmlDeviceGetClockInfo(SM) sampled every 4 ms during each run"
            if nv.h is not None else "NVML unavailable: sm_max_mhz assumed",
            "pipe_warp_inst_per_clk_per_smsp": per_clk,
            "random_sector_g_per_s": rnd, "random_sector_array_bytes": int(min(filter_bytes, 8 << 30))}


def top_roofline(r, kernel, traffic, traffic_src):
    """The line's `roofline` object for the dominant kernel `r` (an entry of `rooflines`): quoted against the measured
    limit that BINDS the kernel (`binds`: the busiest of the instruction limits, the random-sector rate and the streamed
    HBM bytes), with the instruction roofline — both counts, the restated one of DESIGN.md §6 and SURVEY.md §8(d)'s
    planning figure — beside it under "alu"."""
    alu = {"achieved": r["achieved"], "peak": r["peak"], "unit": "Tiop/s", "frac": r["frac"],
           "frac_with_survey_count": r.get("frac_with_survey_count"),
           "ops_per_kmer": sum(r["algorithmic_ops_per_kmer"].values()),
           "survey_ops_per_kmer": r.get("survey_planning_ops_per_kmer"), "peak_source": r["peak_source"]}
    binds = r["binds"]
    if binds == "random_sector":
        rs = r["random_sector"]
        out = {"bound": "hbm", "limit": "random 32-byte sector accesses: DRAM transactions, not bytes, bind (profiles/ceilings_ncu_r02.md)",
               "achieved": rs["achieved_g_per_s"] * 32.0, "peak": rs["ceiling_g_per_s"] * 32.0, "unit": "GB/s",
               "frac": rs["frac"], "peak_source": "measured in this run: %s, x 32 B" % rs["ceiling"]}
    elif binds == "hbm_bytes":
        out = {"bound": "hbm", "limit": "streamed bytes", "achieved": r["hbm"]["achieved"], "peak": r["hbm"]["peak"],
               "unit": "GB/s", "frac": r["hbm"]["frac"], "peak_source": r["hbm"]["peak_source"]}
    else:  # an instruction limit: the algorithmic instruction roofline is the fraction
        out = {"bound": "alu", "limit": binds, "achieved": r["achieved"], "peak": r["peak"], "unit": "Tiop/s",
               "frac": r["frac"], "peak_source": r["peak_source"]}
    out.update({"kernel": kernel, "binds": binds, "binds_busy": r["binds_busy"], "traffic": traffic,
                "traffic_source": traffic_src, "alu": alu, "random_sector": r["random_sector"], "hbm_streaming": r["hbm"]})
    return out


def step_roofline(roof, ms_per_step, pack_bytes, clear_bytes, hbm_gbs):
    """Shortest time one step could take on this box: each fused kernel at the measured limit that binds it
    (its time x the busy fraction of that limit) + the streamed bytes of pack and clear at the HBM rate."""
    t_i = roof["insert_kernel"]["ms"] * min(1.0, roof["insert_kernel"]["binds_busy"])
    t_q = roof["query_kernel"]["ms"] * min(1.0, roof["query_kernel"]["binds_busy"])
    t_s = (pack_bytes + clear_bytes) / (hbm_gbs * 1e9) * 1e3
    return {"roofline_ms": t_i + t_q + t_s, "ms_per_step": ms_per_step, "frac": (t_i + t_q + t_s) / ms_per_step,
            "parts_ms": {"insert_kernel_at_%s" % roof["insert_kernel"]["binds"]: t_i,
                         "query_kernel_at_%s" % roof["query_kernel"]["binds"]: t_q,
                         "pack_and_clear_bytes_at_hbm": t_s},
            "timed": "sbf_clear + sbf_insert_seq/_records + sbf_query_records of one read batch (pack, fused kernels, counts)"}


def alu_roofline(ops, n_units, ms, ceil, clock_mhz, executed, survey_ops=None):
    """Instruction roofline of one kernel.  achieved = ALGORITHMIC lane-ops per second.  peak = the rate the SM
    sub-partitions can issue that algorithmic mix at, from rates measured in this run: per warp of 32 units the
    alu-pipe ops need ops_alu / r_alu clocks PLUS c_wide clocks per wide multiply (the LOP3:IMAD.HI mixes show the
    64-bit-result multiplies serialise with the alu pipe: c_wide = 4 / rate(LOP3:IMAD.HI 3:1) - 3 / r_alu), the
    fma-pipe ops (ops_fma + ops_wide) / r_fma, and all of them together total / r_issue; the slowest binds.
    `executed` (ncu) gives how busy the instructions the kernel really issues keep each of those limits."""
    pr = ceil["pipe_warp_inst_per_clk_per_smsp"]
    r_alu, r_fma, r_issue = pr["LOP3"], pr["IMAD"], pr["LOP3:IMAD 1:1"]
    c_wide = 4.0 / pr["LOP3:IMAD.HI 3:1"] - 3.0 / r_alu if pr.get("LOP3:IMAD.HI 3:1") else 1.0 / r_fma
    wide = ops.get("wide", 0.0)
    total = ops["alu"] + ops["fma"] + wide
    clk_per_unit = max(ops["alu"] / r_alu + wide * c_wide, (ops["fma"] + wide) / r_fma, total / r_issue)  # per warp, per SMSP
    lanes_per_s = 32.0 * N_SMSP * clock_mhz * 1e6
    peak = total / clk_per_unit * lanes_per_s / 1e12                                # T lane-ops/s for this mix
    achieved = total * n_units / (ms * 1e-3) / 1e12
    out = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "Tiop/s", "frac": achieved / peak, "ms": ms,
           "gkmers_s": n_units / ms / 1e6,
           "algorithmic_ops_per_kmer": dict(ops), "peak_source": "measured: pipe rates alu %.3f fma %.3f issue %.3f "
           "warp-inst/clk/SMSP, %.2f clk per wide multiply next to alu work, x %d SMSP x %.0f MHz"
           % (r_alu, r_fma, r_issue, c_wide, N_SMSP, clock_mhz)}
    if survey_ops:
        out["survey_planning_ops_per_kmer"] = survey_ops
        out["frac_with_survey_count"] = survey_ops * n_units / (ms * 1e-3) / 1e12 / (lanes_per_s * r_alu / 1e12)
    if executed:
        cyc = ms * 1e-3 * clock_mhz * 1e6 * N_SMSP                                   # SMSP-cycles of the launch
        scale = n_units / executed["units"]        # the capture's counts, scaled to this launch's number of k-mers
        busy = {"alu_pipe": executed["inst_alu"] * scale / r_alu / cyc, "fma_pipe": executed["inst_fma"] * scale / r_fma / cyc,
                "issue": executed["inst_total"] * scale / r_issue / cyc}
        out["executed_warp_inst_per_kmer"] = {k[5:]: v * 32.0 / executed["units"] for k, v in executed.items()
                                              if k.startswith("inst_")}
        out["busy_fraction_of_measured_limit"] = busy
        out["binding_instruction_limit"] = max(busy, key=busy.get)
    return out


def cpu_baseline(args, w):
    import oracle
    p = w.params
    ins_bases = min(w.insert_bases.size, args.ref_insert_bases)
    n_reads = min(max(w.n_reads, 1), args.ref_reads)
    seq_s, reads_s, offs_s = make_oracle_sample(w, ins_bases, n_reads)
    o = oracle.OracleSBF(p["k"], p["m"], p["s"], p["H"], p["num_bits"])
    sample = "insert first %d bases of the %s sequence + query first %d reads x %d, filter %d bits" % (
        ins_bases, args.workload, n_reads, w.read_len, o.num_bits)
    a, b, ti, tq = oracle_sample_step(o, seq_s, reads_s, offs_s, False)
    single = {"value": (a + b) / (ti + tq) / 1e9, "insert": a / ti / 1e9, "query": b / tq / 1e9}
    a, b, ti, tq = oracle_sample_step(o, seq_s, reads_s, offs_s, True)
    cores = oracle.num_threads()
    return ({"value": (a + b) / (ti + tq) / 1e9, "unit": "G k-mers/s", "cores": cores, "kind": "oracle",
             "sample": sample, "insert_gkmers_s": a / ti / 1e9, "query_gkmers_s": b / tq / 1e9,
             "timed": "insert + query of the sample (the filter is cleared before the clock starts)",
             "single_thread": single}, (seq_s, reads_s, offs_s), oracle_sample_step.last_counts)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="config3", choices=["config1", "config2", "config3", "config4"])
    ap.add_argument("--scale", type=float, default=1.0, help="shrink the workload (tests only)")
    ap.add_argument("--read-batch", type=int, default=4_000_000, help="reads per query batch (one per step)")
    ap.add_argument("--batches", type=int, default=4, help="distinct read batches rotated over the steps")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ref-scale", type=float, default=0.1, help="--impl reference: sequence generated at this scale")
    ap.add_argument("--ref-insert-bases", type=int, default=10_000_000)
    ap.add_argument("--ref-reads", type=int, default=50_000)
    args = ap.parse_args()
    if args.steps < 1 or args.warmup < 0:
        raise SystemExit("need --steps >= 1, --warmup >= 0")
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())

"""Parameter sweep of BASELINE.json config 5 and the FPR-vs-size experiment.

    python -m paper_2606_24417_b200.sweep [--scale 1.0] [--reads 2000000] [--points cross|axes]
                                          [--sizes 28 34] [--out profiles/sweep_r02.md]

For every (s, m, H) point at k = 31 it creates a filter, inserts the config-3 sequence, queries one batch of
config-3 reads, and reports insert / query G k-mers/s (CUDA events around the library calls, best of 3),
the measured FPR on the uniform-random reads (odd read index: aliens; expected true members are below
1e-8 relative, P:389-397 uses the same definition), the hit rate of the sampled reads, the effective
bits per inserted k-mer, and the Pareto set of (FPR, time).  Then the size sweep (Fig. 6 of the paper,
P:389-397) for s in {28, 30, 31}.  Everything runs through the C ABI; the oracle is not involved
(tests/ pins the bits; this tool only reports statistics).  Inputs: seeded synthetic (seqgen/).
The FPR-vs-size experiment proper (10^9 random 31-mers, 2^22 .. 2^39 bits) is paper_2606_24417_b200/fpr_size.py.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

_ACGT = np.zeros(256, dtype=bool)
for _c in b"ACGTacgt":
    _ACGT[_c] = True


def _valid_windows(seq: np.ndarray, k: int) -> int:
    """Number of length-k windows of one sequence without a non-ACGT symbol (bookkeeping for the rates)."""
    n, total, step = seq.size, 0, 1 << 26
    for a in range(0, max(n - k + 1, 0), step):
        e = min(a + step + k - 1, n)
        bad = ~_ACGT[seq[a:e]]
        if not bad.any():
            total += e - a - k + 1
        else:
            cs = np.concatenate(([0], np.cumsum(bad, dtype=np.int32)))
            total += int(np.count_nonzero(cs[k:] - cs[:-k] == 0))
    return total


def _valid_per_read(reads: np.ndarray, read_len: int, k: int) -> np.ndarray:
    n = reads.size // read_len
    out = np.full(n, max(read_len - k + 1, 0), dtype=np.int64)
    for r in np.flatnonzero((~_ACGT[reads]).reshape(n, read_len).any(axis=1)):
        out[r] = _valid_windows(reads[r * read_len:(r + 1) * read_len], k)
    return out


def run_point(sbf, torch, k, m, s, H, num_bits, d_seq, n_ins, d_reads, d_offs, n_reads, read_len, valid, reps=3):
    f = sbf.sbf_create(k, m, s, H, num_bits)
    try:
        sbf.sbf_reserve(f, max(d_seq.numel(), d_reads.numel()))
        bm = torch.empty((d_reads.numel() + 31) // 32, dtype=torch.int32, device="cuda")
        hc = torch.empty(n_reads, dtype=torch.int32, device="cuda")
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t_ins, t_q = [], []
        for _ in range(reps):
            sbf.sbf_clear(f)
            e0.record()
            sbf.sbf_insert_seq(f, d_seq, d_seq.numel())
            e1.record(); e1.synchronize()
            t_ins.append(e0.elapsed_time(e1))
        for _ in range(reps):
            e0.record()
            sbf.sbf_query_records(f, d_reads, d_offs, n_reads, d_reads.numel(), bm, hc)
            e1.record(); e1.synchronize()
            t_q.append(e0.elapsed_time(e1))
        cnt = hc.cpu().numpy().view(np.uint32).astype(np.int64)
        return {
            "k": k, "m": m, "s": s, "H": H, "log2_bits": int(np.log2(sbf.sbf_num_bits(f))),
            "specialized": bool(sbf.sbf_is_specialized(f)),
            "bits_per_kmer": sbf.sbf_num_bits(f) / max(1, n_ins),
            "insert_gkmers_s": n_ins / min(t_ins) / 1e6, "query_gkmers_s": int(valid.sum()) / min(t_q) / 1e6,
            "insert_ms": min(t_ins), "query_ms": min(t_q),
            "fpr_random": float(cnt[1::2].sum()) / max(1, int(valid[1::2].sum())),
            "hit_sampled": float(cnt[0::2].sum()) / max(1, int(valid[0::2].sum())),
        }
    finally:
        sbf.sbf_destroy(f)


def pareto(points, keys=("fpr_random", "time_ms")):
    """Indices of the points no other point beats on every key (lower is better)."""
    out = []
    for i, p in enumerate(points):
        dominated = any(all(q[x] <= p[x] for x in keys) and any(q[x] < p[x] for x in keys)
                        for j, q in enumerate(points) if j != i)
        if not dominated:
            out.append(i)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--scale", type=float, default=1.0, help="fraction of the 250 Mbp config-3 sequence")
    ap.add_argument("--reads", type=int, default=2_000_000)
    ap.add_argument("--points", default="cross", choices=["cross", "axes"])
    ap.add_argument("--sizes", type=int, nargs=2, default=[28, 34], help="log2 of the smallest / largest filter size in bits")
    ap.add_argument("--out", default=None, help="markdown summary; the full table goes to <out minus .md>.csv")
    args = ap.parse_args()

    import torch
    import seqgen
    import paper_2606_24417_b200 as sbf
    if not torch.cuda.is_available():
        raise SystemExit("sweep: no CUDA device (there is no CPU fallback)")
    k = 31
    w = seqgen.config3(scale=args.scale, n_reads=args.reads)
    reads = w.read_batch(0, args.reads)
    valid = _valid_per_read(reads, w.read_len, k)
    n_ins = _valid_windows(w.insert_bases, k)
    d_seq = torch.from_numpy(w.insert_bases).cuda()
    d_reads = torch.from_numpy(reads).cuda()
    d_offs = torch.from_numpy(seqgen.fixed_offsets(args.reads, w.read_len).view(np.int64)).cuda()
    common = (d_seq, n_ins, d_reads, d_offs, args.reads, w.read_len, valid)

    # BASELINE.json configs[4]: the (s, m, H) cross product at EVERY filter size 2^28 .. 2^34
    rows = []
    for lb in range(args.sizes[0], args.sizes[1] + 1):
        for (s, m, H) in seqgen.config5_points(full_cross=(args.points == "cross")):
            r = run_point(sbf, torch, k, m, s, H, 1 << lb, *common)
            r["time_ms"] = r["insert_ms"] + r["query_ms"]
            r["gkmers_s"] = (n_ins + int(valid.sum())) / r["time_ms"] / 1e6       # insert + query throughput of the point
            rows.append(r)
            print(json.dumps(r), flush=True)
    # Pareto set of (FPR, bits per k-mer, throughput): lower FPR, fewer bits, less time per pass
    front = set(pareto(rows, keys=("fpr_random", "bits_per_kmer", "time_ms")))

    if args.out:
        base = args.out[:-3] if args.out.endswith(".md") else args.out
        with open(base + ".csv", "w") as fh:
            fh.write("log2_bits,bits_per_kmer,s,m,H,kernel,insert_gkmers_s,query_gkmers_s,step_gkmers_s,fpr_random,hit_sampled,pareto\n")
            for i, r in enumerate(rows):
                fh.write("%d,%.3f,%d,%d,%d,%s,%.2f,%.2f,%.2f,%.4e,%.5f,%d\n" % (
                    r["log2_bits"], r["bits_per_kmer"], r["s"], r["m"], r["H"], "spec" if r["specialized"] else "rt",
                    r["insert_gkmers_s"], r["query_gkmers_s"], r["gkmers_s"], r["fpr_random"], r["hit_sampled"], int(i in front)))
        with open(args.out if args.out.endswith(".md") else base + ".md", "w") as fh:
            fh.write("# BASELINE config 5: (s, m, H) cross product x filter sizes (k = 31, synthetic config-3 sequence and reads)\n\n")
            fh.write("Command: `python -m paper_2606_24417_b200.sweep %s`\n\n" % " ".join(sys.argv[1:]))
            fh.write("%d inserted k-mers, %d reads x %d (%d valid query k-mers, half of them aliens). %d points = %d (s, m, H) x "
                     "filter sizes 2^%d .. 2^%d bits; all of them in `%s`. Rates are whole library calls (pack + fused kernel "
                     "+ counts), best of 3, device-resident input; FPR = positives among the k-mers of the uniform-random reads; "
                     "bits per k-mer = effective filter bits / inserted k-mers.\n\n" % (
                         n_ins, args.reads, w.read_len, int(valid.sum()), len(rows),
                         len(rows) // (args.sizes[1] - args.sizes[0] + 1), args.sizes[0], args.sizes[1], os.path.basename(base + ".csv")))
            fh.write("## Pareto set of (FPR, bits per k-mer, throughput): %d of %d points\n\n" % (len(front), len(rows)))
            fh.write("| log2 bits | bits / k-mer | s | m | H | insert G k-mers/s | query G k-mers/s | FPR |\n|---|---|---|---|---|---|---|---|\n")
            for i in sorted(front, key=lambda i: (rows[i]["log2_bits"], rows[i]["fpr_random"])):
                r = rows[i]
                fh.write("| %d | %.2f | %d | %d | %d | %.1f | %.1f | %.3e |\n" % (
                    r["log2_bits"], r["bits_per_kmer"], r["s"], r["m"], r["H"], r["insert_gkmers_s"], r["query_gkmers_s"], r["fpr_random"]))
            hs = sorted({r["H"] for i, r in enumerate(rows) if i in front})
            fh.write("\nH values on the Pareto set: %s (the paper: all Pareto points at H = 4, P:359).\n" % hs)
            fh.write("\n## The one-factor axes through (28, 16, 4), per filter size\n\n")
            fh.write("| log2 bits | s | m | H | insert G k-mers/s | query G k-mers/s | FPR | hit rate (sampled reads) |\n|---|---|---|---|---|---|---|---|\n")
            for r in rows:
                if sum((r["s"] != 28, r["m"] != 16, r["H"] != 4)) <= 1:
                    fh.write("| %d | %d | %d | %d | %.1f | %.1f | %.3e | %.4f |\n" % (
                        r["log2_bits"], r["s"], r["m"], r["H"], r["insert_gkmers_s"], r["query_gkmers_s"], r["fpr_random"], r["hit_sampled"]))
    return 0


if __name__ == "__main__":
    sys.exit(main())

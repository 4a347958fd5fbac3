"""Parameter sweep of BASELINE.json config 5 and the FPR-vs-size experiment.

    python -m paper_2606_24417_b200.sweep [--scale 1.0] [--reads 2000000] [--points cross|axes]
                                          [--log2-bits 32] [--sizes 28 34] [--out profiles/sweep_r01.md]

For every (s, m, H) point at k = 31 it creates a filter, inserts the config-3 sequence, queries one batch of
config-3 reads, and reports insert / query G k-mers/s (CUDA events around the library calls, best of 3),
the measured FPR on the uniform-random reads (odd read index: aliens; expected true members are below
1e-8 relative, P:389-397 uses the same definition), the hit rate of the sampled reads, the effective
bits per inserted k-mer, and the Pareto set of (FPR, time).  Then the size sweep (Fig. 6 of the paper,
P:389-397) for s in {28, 30, 31}.  Everything runs through the C ABI; the oracle is not involved
(tests/ pins the bits; this tool only reports statistics).  Inputs: seeded synthetic (seqgen/).
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
    ap.add_argument("--log2-bits", type=int, default=32)
    ap.add_argument("--sizes", type=int, nargs=2, default=[28, 34])
    ap.add_argument("--out", default=None)
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

    rows = []
    for (s, m, H) in seqgen.config5_points(full_cross=(args.points == "cross")):
        r = run_point(sbf, torch, k, m, s, H, 1 << args.log2_bits, *common)
        r["time_ms"] = r["insert_ms"] + r["query_ms"]
        rows.append(r)
        print(json.dumps(r), flush=True)
    front = set(pareto(rows))
    sizes = []
    for lb in range(args.sizes[0], args.sizes[1] + 1):
        for s in (28, 30, 31):
            r = run_point(sbf, torch, k, 16, s, 4, 1 << lb, *common)
            sizes.append(r)
            print(json.dumps(r), flush=True)

    if args.out:
        with open(args.out, "w") as fh:
            fh.write("# Config 5 sweep and FPR vs filter size (k = 31, synthetic config-3 sequence and reads)\n\n")
            fh.write("Command: `python -m paper_2606_24417_b200.sweep %s`\n\n" % " ".join(sys.argv[1:]))
            fh.write("%d inserted k-mers, %d reads x %d (%d valid query k-mers, half of them aliens). Rates are whole library "
                     "calls (pack + fused kernel + counts), best of 3, device-resident input. `spec` = specialised streaming "
                     "kernels; `rt` = runtime-parameter kernel (Alg. 1/2 as printed, every k-mer recomputed).\n\n" %
                     (n_ins, args.reads, w.read_len, int(valid.sum())))
            fh.write("## (s, m, H) at 2^%d bits (%.1f bits per inserted k-mer)\n\n" % (args.log2_bits, rows[0]["bits_per_kmer"]))
            fh.write("| s | m | H | kernel | insert G k-mers/s | query G k-mers/s | FPR (random reads) | hit rate (sampled reads) | Pareto (FPR, time) |\n")
            fh.write("|---|---|---|---|---|---|---|---|---|\n")
            for i, r in enumerate(rows):
                fh.write("| %d | %d | %d | %s | %.1f | %.1f | %.3e | %.4f | %s |\n" % (
                    r["s"], r["m"], r["H"], "spec" if r["specialized"] else "rt", r["insert_gkmers_s"], r["query_gkmers_s"],
                    r["fpr_random"], r["hit_sampled"], "yes" if i in front else ""))
            fh.write("\n## FPR vs filter size, (m, H) = (16, 4)\n\n| log2 bits | bits / k-mer | s | insert G k-mers/s | query G k-mers/s | FPR |\n|---|---|---|---|---|---|\n")
            for r in sizes:
                fh.write("| %d | %.2f | %d | %.1f | %.1f | %.3e |\n" % (r["log2_bits"], r["bits_per_kmer"], r["s"],
                                                                   r["insert_gkmers_s"], r["query_gkmers_s"], r["fpr_random"]))
    return 0


if __name__ == "__main__":
    sys.exit(main())

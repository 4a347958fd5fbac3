"""FPR versus filter size (§V-D, Fig. 6), on synthetic stand-ins.

    python -m paper_2606_24417_b200.fpr_size [--kmers 1000000000] [--sizes 22 39] [--s 28 30 31] [--scale 1.0]
                                             [--out profiles/fpr_size_r02.md]

The paper inserts the C. elegans reference and counts the false positives among 10^9 random 31-mers while the filter
grows from 2^22 to 2^39 bits, for s in {28, 30, 31} (k = 31, m = 16, H = 4).  That reference is not available offline:
the inserted sequence here is the seeded config-3 sequence (250 Mbp order-5 Markov with N runs, seqgen/), and the 10^9
aliens are 10^9 records of 31 uniform bases — record r is symbols [31 r, 31 r + 31) of the stream seqgen.uniform(seed,
.) — generated ON THE DEVICE batch by batch (seqgen.uniform_device; 31 GB of symbols never cross PCIe) and queried
through sbf_query_records (one k-mer per record).  Among 10^9 uniform 31-mers the expected number of true members of a
2.5e8-k-mer set is 10^9 * 2.5e8 / 4^31 < 1e-1, so every positive counts as a false positive (the paper's definition).

Everything runs through the C ABI; the oracle is not involved here (tests/test_gpu_fpr_size.py compares the same
device-generated records with the oracle, bit for bit, on a 10^6-record slice).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

K, M, H = 31, 16, 4
ALIEN_SEED = 6


def count_false_positives(sbf, torch, seqgen, handle, n_kmers, batch, d_offs, d_bases, d_bitmap, d_counts):
    """Positives among records [0, n_kmers) of the alien stream; also the positives among the first 10^6."""
    total, first_million = 0, 0
    for first in range(0, n_kmers, batch):
        n = min(batch, n_kmers - first)
        seqgen.uniform_device(ALIEN_SEED, first * K, n * K, out=d_bases)
        sbf.sbf_query_records(handle, d_bases, d_offs, n, n * K, d_bitmap, d_counts)
        c = d_counts[:n]
        total += int(c.sum(dtype=torch.int64).item())
        if first < 1_000_000:
            first_million += int(c[:min(n, 1_000_000 - first)].sum(dtype=torch.int64).item())
    return total, first_million


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--kmers", type=int, default=1_000_000_000)
    ap.add_argument("--sizes", type=int, nargs=2, default=[22, 39], help="log2 of the smallest and largest filter size in bits")
    ap.add_argument("--s", type=int, nargs="+", default=[28, 30, 31])
    ap.add_argument("--scale", type=float, default=1.0, help="fraction of the 250 Mbp config-3 sequence to insert")
    ap.add_argument("--batch", type=int, default=1 << 25, help="31-mers per query batch")
    ap.add_argument("--out", default=None)
    args = ap.parse_args()

    import torch
    import seqgen
    import paper_2606_24417_b200 as sbf
    if not torch.cuda.is_available():
        raise SystemExit("fpr_size: no CUDA device (there is no CPU fallback)")
    from paper_2606_24417_b200.sweep import _valid_windows

    w = seqgen.config3(scale=args.scale)
    n_ins = _valid_windows(w.insert_bases, K)
    d_seq = torch.from_numpy(w.insert_bases).cuda()
    batch = min(args.batch, args.kmers)
    d_offs = (torch.arange(batch + 1, dtype=torch.int64, device="cuda") * K)
    d_bases = torch.empty(batch * K, dtype=torch.uint8, device="cuda")
    d_bitmap = torch.empty((batch * K + 31) // 32, dtype=torch.int32, device="cuda")
    d_counts = torch.empty(batch, dtype=torch.int32, device="cuda")
    free_b, _ = torch.cuda.mem_get_info()

    rows = []
    for lb in range(args.sizes[0], args.sizes[1] + 1):
        if (1 << lb) // 8 > free_b - (2 << 30):
            print(json.dumps({"log2_bits": lb, "skipped": "filter does not fit the free device memory"}), flush=True)
            continue
        for s in args.s:
            t0 = time.perf_counter()
            f = sbf.sbf_create(K, M, s, H, 1 << lb)
            try:
                sbf.sbf_reserve(f, max(d_seq.numel(), batch * K))
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                sbf.sbf_insert_seq(f, d_seq, d_seq.numel())
                e1.record()
                fp, fp1m = count_false_positives(sbf, torch, seqgen, f, args.kmers, batch, d_offs, d_bases, d_bitmap, d_counts)
                torch.cuda.synchronize()
                r = {"log2_bits": lb, "s": s, "bits_per_kmer": (1 << lb) / max(1, n_ins), "kmers": args.kmers,
                     "false_positives": fp, "fpr": fp / args.kmers, "fp_first_1e6": fp1m,
                     "insert_ms": e0.elapsed_time(e1), "wall_s": time.perf_counter() - t0}
            finally:
                sbf.sbf_destroy(f)
            rows.append(r)
            print(json.dumps(r), flush=True)

    if args.out:
        with open(args.out, "w") as fh:
            fh.write("# FPR vs filter size (PAPER.md:389-397, Fig. 6) on synthetic stand-ins\n\n")
            fh.write("Command: `python -m paper_2606_24417_b200.fpr_size %s`\n\n" % " ".join(sys.argv[1:]))
            fh.write("Inserted: the config-3 sequence (%d valid 31-mers; stand-in for the C. elegans reference, which is not "
                     "available offline). Queried: %d records of 31 uniform bases generated on the device "
                     "(`seqgen.uniform_device(seed %d)`), all of them aliens (expected true members < 0.1). k = 31, m = 16, "
                     "H = 4. The paper's ordering FPR(s=28) < FPR(s=30) < FPR(s=31) (PAPER.md:389) is reproduced wherever the "
                     "counts are above noise; its absolute values belong to another sequence and are not comparable.\n\n"
                     % (n_ins, args.kmers, ALIEN_SEED))
            fh.write("| log2 bits | bits per inserted k-mer | " + " | ".join("FP s=%d | FPR s=%d" % (s, s) for s in args.s) + " |\n")
            fh.write("|---|---|" + "---|---|" * len(args.s) + "\n")
            for lb in sorted({r["log2_bits"] for r in rows}):
                rr = {r["s"]: r for r in rows if r["log2_bits"] == lb}
                fh.write("| %d | %.3g | " % (lb, next(iter(rr.values()))["bits_per_kmer"]) +
                         " | ".join("%d | %.3e" % (rr[s]["false_positives"], rr[s]["fpr"]) if s in rr else " | " for s in args.s) + " |\n")
            fh.write("\nFirst 10^6 records (the slice `tests/test_gpu_fpr_size.py` compares with the oracle bit for bit on a "
                     "reduced sequence): " + ", ".join("2^%d/s=%d: %d" % (r["log2_bits"], r["s"], r["fp_first_1e6"])
                                                       for r in rows if r["log2_bits"] in (26, 30, 32)) + "\n")
    return 0


if __name__ == "__main__":
    sys.exit(main())

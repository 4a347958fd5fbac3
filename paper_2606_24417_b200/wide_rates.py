"""Rates of the WIDE path: protein and DNA-triplet alphabets and DNA k-mers of more
than 32 bases, with and without a specialised streaming instance.

    python -m paper_2606_24417_b200.wide_rates [--bytes 60000000] [--bits 32] [--out profiles/wide_r02.md]

The paper gives no workload for these ("larger alphabets remain functional"): the inputs are seeded
uniform symbols (seqgen/), one sequence of --bytes bytes; it is inserted, queried as one sequence (every k-mer a member)
and queried again cut into 150-byte records.  Device-resident input, kernel time from sbf_get_timing (CUDA events around
the fused kernel), best of 4.  Everything runs through the C ABI; parity of these very paths against the oracle is
tests/test_gpu_wide.py.
"""
from __future__ import annotations

import argparse
import json
import os
import string
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

DNA, PROTEIN, TRIPLET = 0, 1, 2
# (label, alphabet, k, m, s, H)
CASES = [("protein k=12", PROTEIN, 12, 6, 10, 4), ("protein k=25", PROTEIN, 25, 7, 20, 4),
         ("DNA triplets k=10", TRIPLET, 10, 5, 8, 4), ("DNA triplets k=21", TRIPLET, 21, 9, 18, 6),
         ("DNA k=63, no instance", DNA, 63, 30, 59, 4), ("DNA k=63, instance (63,31,60,4)", DNA, 63, 31, 60, 4),
         ("DNA k=33, instance (33,16,30,4)", DNA, 33, 16, 30, 4)]


def protein_text(seqgen, seed, n):
    """Seeded uniform bases mapped to the 26 letters (three bases -> one letter index mod 26)."""
    aa = np.frombuffer(string.ascii_uppercase.encode(), dtype=np.uint8)
    r = seqgen.uniform(seed, 3 * n).astype(np.int64).reshape(n, 3)
    return aa[((((r[:, 0] >> 1) & 3) * 16 + ((r[:, 1] >> 1) & 3) * 4 + ((r[:, 2] >> 1) & 3)) % 26)].copy()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--bytes", type=int, default=60_000_000)
    ap.add_argument("--bits", type=int, default=32, help="log2 of the filter size in bits")
    ap.add_argument("--out", default=None)
    args = ap.parse_args()
    import torch
    import seqgen
    import paper_2606_24417_b200 as sbf

    torch.cuda.set_device(0)
    n, rec_len = args.bytes, 150
    n_rec = n // rec_len
    d_offs = torch.arange(0, n_rec + 1, dtype=torch.int64, device="cuda") * rec_len
    d_bm = torch.empty((n + 31) // 32, dtype=torch.int32, device="cuda")
    d_hc = torch.empty(n_rec, dtype=torch.int32, device="cuda")
    texts = {PROTEIN: protein_text(seqgen, 5, n), DNA: seqgen.uniform(8, n), TRIPLET: seqgen.uniform(7, n)}
    rows = []
    for label, alpha, k, m, s, H in CASES:
        nb = 3 if alpha == TRIPLET else 1
        d = torch.from_numpy(texts[alpha]).cuda()
        with sbf.SuperBloomFilter(k=k, m=m, s=s, H=H, num_bits=1 << args.bits, alphabet=alpha) as f:
            sbf.sbf_set_timing(f.handle, True)
            ti, tq, tr = [], [], []
            for _ in range(4):
                f.clear()
                f.insert_seq(d)
                ti.append(sbf.sbf_get_timing(f.handle)[1])
                f.query_seq(d, d_bm)
                tq.append(sbf.sbf_get_timing(f.handle)[1])
                sbf.sbf_query_records(f.handle, d, d_offs, n_rec, n_rec * rec_len, d_bm, d_hc)
                tr.append(sbf.sbf_get_timing(f.handle)[1])
            torch.cuda.synchronize()
            hits = int(d_hc.sum(dtype=torch.int64).item())
            nk = n // nb - k + 1
            nkr = n_rec * (rec_len // nb - k + 1)
            assert hits == nkr, "every k-mer of an inserted sequence must be reported present (PAPER.md:90)"
            rows.append(dict(case=label, k=k, m=m, s=s, H=H, specialised=bool(f.specialized),
                             insert_ms=min(ti), query_seq_ms=min(tq), query_records_ms=min(tr),
                             insert_gkmers_s=nk / min(ti) / 1e6, query_seq_gkmers_s=nk / min(tq) / 1e6,
                             query_records_gkmers_s=nkr / min(tr) / 1e6))
            print(json.dumps(rows[-1]), flush=True)
    if args.out:
        lines = ["# Rates of the wide path: other alphabets and DNA k > 32 (round 2)", "",
                 "Command: `python -m paper_2606_24417_b200.wide_rates --out %s`" % args.out, "",
                 "%d bytes of seeded uniform symbols, filter 2^%d bits; kernel time (CUDA events, `sbf_get_timing`), best of 4; "
                 "G k-mers/s. Runtime-parameter shapes run `wide_tile_kernel`; \"instance\" rows run the specialised streaming "
                 "kernels (`csrc/sbf_inst_wide.cu`). Every k-mer of the inserted sequence is reported present in each run."
                 % (n, args.bits), "",
                 "| case | (k, m, s, H) | kernel | insert | query, one sequence | query, 150-byte records |", "|---|---|---|---|---|---|"]
        for r in rows:
            lines.append("| %s | (%d, %d, %d, %d) | %s | %.1f | %.1f | %.1f |" % (
                r["case"], r["k"], r["m"], r["s"], r["H"], "streaming instance" if r["specialised"] else "`wide_tile_kernel`",
                r["insert_gkmers_s"], r["query_seq_gkmers_s"], r["query_records_gkmers_s"]))
        os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)
        with open(args.out, "w") as fh:
            fh.write("\n".join(lines) + "\n")
    return 0


if __name__ == "__main__":
    sys.exit(main())

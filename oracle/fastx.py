"""Plain line-by-line FASTA / FASTQ reader for the oracle side (TEST INFRASTRUCTURE, NOT PRODUCT).

What the product's device-side normaliser (paper_2606_24417_b200/csrc/sbf_fastx.cuh) must reproduce, written the slow,
obvious way with bytes.split ("consecutive records are concatenated").  Text rules (as
stated in include/sbf.h): lines end at '\\n'; '\\r' is dropped; every other byte of a sequence line is kept verbatim.
  FASTA  a line whose first byte is '>' is a header and starts a record; every other line belongs to the current
         record; text before the first header is the `pre` segment (inserted by the insert call, ignored by queries).
  FASTQ  four lines per record: header, sequence, '+', quality (line index mod 4); a record starts at a line with
         index 0 mod 4 whose first byte is neither '\\n' nor '\\r' (A23: a blank line, e.g. the one a
         text ending in two newlines has, still counts as a line but opens no record).
Shares nothing with the CUDA path and never imports it.
"""
from __future__ import annotations

import numpy as np

FASTA, FASTQ = 1, 2


def detect(text: bytes) -> int:
    for c in text:
        if c not in b"\n\r ":
            return FASTQ if c == ord("@") else FASTA
    return FASTA


def parse(text: bytes, fmt: int = 0):
    """-> (pre: bytes, records: list of bytes).  `pre` is empty for FASTQ."""
    if fmt == 0:
        fmt = detect(text)
    lines = text.split(b"\n")
    pre, records = bytearray(), []
    if fmt == FASTA:
        for raw in lines:
            if raw.startswith(b">"):
                records.append(bytearray())
            else:
                (records[-1] if records else pre).extend(raw.replace(b"\r", b""))
    else:
        for idx, raw in enumerate(lines):
            if idx % 4 == 0:
                if raw[:1] not in (b"", b"\r"):
                    records.append(bytearray())
            elif idx % 4 == 1:
                if records:
                    records[-1].extend(raw.replace(b"\r", b""))
    return bytes(pre), [bytes(r) for r in records]


def dense(text: bytes, fmt: int = 0, with_pre: bool = True):
    """-> (bases uint8[total], offsets uint64[n+1]) of the dense record batch; with_pre puts the text before the first
    FASTA header in front as a record of its own (what the insert call inserts)."""
    pre, records = parse(text, fmt)
    recs = ([pre] if with_pre and pre else []) + records
    lens = np.array([len(r) for r in recs], dtype=np.uint64)
    offsets = np.concatenate(([0], np.cumsum(lens))).astype(np.uint64)
    bases = np.frombuffer(b"".join(recs), dtype=np.uint8).copy() if recs else np.zeros(0, dtype=np.uint8)
    return bases, offsets

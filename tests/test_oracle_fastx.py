"""The oracle-side FASTA / FASTQ reader (oracle/fastx.py) on literal texts whose records are written out by hand."""
import numpy as np

from oracle import fastx
import seqgen


def test_fasta_literal():
    text = b"ACG\nT\r\n>r1 desc\nAAAA\nCC\n\n>r2\n>r3\r\nGG>T\nN\n"
    pre, recs = fastx.parse(text)
    assert pre == b"ACGT" and recs == [b"AAAACC", b"", b"GG>TN"]
    bases, offs = fastx.dense(text)
    assert bases.tobytes() == b"ACGTAAAACCGG>TN" and offs.tolist() == [0, 4, 10, 10, 15]
    bases, offs = fastx.dense(text, with_pre=False)
    assert bases.tobytes() == b"AAAACCGG>TN" and offs.tolist() == [0, 6, 6, 11]
    assert fastx.detect(text) == fastx.FASTA and fastx.detect(b"\n\n@x\nA\n+\nI\n") == fastx.FASTQ


def test_fastq_literal():
    text = b"@a\nACGT\n+\nIIII\n@b\r\nGG\r\n+\r\n>@\r\n@c\n\n+\n\n@d\nT"
    pre, recs = fastx.parse(text)
    assert pre == b"" and recs == [b"ACGT", b"GG", b"", b"T"]
    assert fastx.dense(text)[1].tolist() == [0, 4, 6, 6, 7]
    assert fastx.parse(b"@a\nAC\n+\nII\n")[1] == [b"AC"]          # the text may end with or without a newline
    assert fastx.parse(b"@a\nAC\n+\nII")[1] == [b"AC"]


def test_fastq_blank_lines_open_no_record():
    """DESIGN.md A23: a line of index 0 mod 4 whose first byte is a line end still counts as a line but starts no record
    (a text that ends in two newlines has no extra empty record)."""
    assert fastx.parse(b"@a\nAC\n+\nII\n\n")[1] == [b"AC"]
    assert fastx.parse(b"@a\nAC\n+\nII\n\n\n\n")[1] == [b"AC"]
    assert fastx.parse(b"@a\r\nAC\r\n+\r\nII\r\n\r\n")[1] == [b"AC"]
    assert fastx.dense(b"@a\nAC\n+\nII\n\n")[1].tolist() == [0, 2]
    # a blank line BETWEEN records shifts the four-line grid (not valid FASTQ; the rule is only that both sides agree):
    # line 4 is blank -> no start, line 5 "@b" is then a sequence line of record a, line 8 "II" starts a record whose
    # sequence line (line 9) is empty
    assert fastx.parse(b"@a\nAC\n+\nII\n\n@b\nGG\n+\nII\n")[1] == [b"AC@b", b""]


def test_generators_round_trip():
    recs = [seqgen.uniform(1, 130), seqgen.uniform(2, 0), seqgen.uniform(3, 61), seqgen.uniform(4, 60)]
    for crlf in (False, True):
        for width in (1, 60, 61, 1000):
            assert fastx.parse(seqgen.fasta_text(recs, width, crlf))[1] == [r.tobytes() for r in recs]
        assert fastx.parse(seqgen.fastq_text(recs, crlf))[1] == [r.tobytes() for r in recs]
        assert fastx.parse(seqgen.fastq_text(recs, crlf, final_newline=False))[1] == [r.tobytes() for r in recs]

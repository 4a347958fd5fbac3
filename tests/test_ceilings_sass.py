"""The pipe-rate micro-benchmarks behind bench.py's ALU roofline are counted in SASS ("a micro-benchmark
counted in SASS instructions"): disassemble the built object and check that the loop body of every
pipe_rate_kernel<MODE> is N x the opcode(s) its mode name promises, in the promised ratio, and next to nothing else.
Runs without a GPU (nvcc cross-compiles, cuobjdump disassembles)."""
import collections
import os
import re
import shutil
import subprocess

import pytest

from paper_2606_24417_b200 import build as B

# per loop iteration (kPipeChains * kPipeUnroll = 256 instructions): expected count of each measured opcode
EXPECT = {
    0: {"LOP3": 256}, 1: {"IMAD": 256}, 2: {"SHF": 256},
    3: {"LOP3": 128, "IMAD": 128}, 4: {"LOP3": 192, "IMAD": 64}, 5: {"LOP3": 224, "IMAD": 32},
    6: {"LOP3": 128, "SHF": 128}, 7: {"IDP": 256}, 8: {"LOP3": 128, "IDP": 128},
    9: {"IMAD": 256}, 10: {"LOP3": 128, "IMAD": 128}, 11: {"PRMT": 256}, 12: {"LOP3": 192, "IMAD": 64},
}


def _histograms():
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    B.build()
    obj = os.path.join(B.OBJDIR, "sbf_bench.o")
    if not os.path.exists(obj):  # a shipped library without its objects (build() had nothing to do)
        B.build(force=True)
    sass = subprocess.run([cuobjdump, "-sass", obj], stdout=subprocess.PIPE, text=True, check=True).stdout
    hist, fn = collections.defaultdict(collections.Counter), None
    for ln in sass.splitlines():
        m = re.search(r"Function : (\S+)", ln)
        if m:
            fn = m.group(1)
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_]+)", ln)
        if m and fn:
            hist[fn][m.group(1)] += 1
    return hist


def test_pipe_rate_loop_bodies_are_counted_in_sass():
    hist = _histograms()
    seen = 0
    for fn, h in hist.items():
        m = re.search(r"pipe_rate_kernelILi(\d+)E", fn)
        if not m:
            continue
        mode = int(m.group(1))
        exp = EXPECT[mode]
        seen += 1
        # ptxas may unroll the outer loop: the body appears `mult` times (plus a remainder loop)
        ok = False
        for mult in range(1, 33):
            if all(0 <= h[op] - mult * n <= 24 for op, n in exp.items()):
                ok = True
                measured = mult * sum(exp.values())
                break
        assert ok, "mode %d: opcode counts %r do not match %r x n" % (mode, dict(h), exp)
        others = sum(h.values()) - measured
        assert others <= 0.06 * measured + 80, "mode %d: %d instructions besides the %d measured ones" % (mode, others, measured)
    assert seen == len(EXPECT)


def test_random_sector_kernels_issue_the_named_access():
    hist = _histograms()
    want = {0: "REDG", 1: "REDG", 2: "LDG", 3: "LDGSTS", 4: "UBLKRED", 5: "LDG", 6: "LDGSTS", 7: "STG"}
    for fn, h in hist.items():
        m = re.search(r"random_sector_kernelILi(\d+)E", fn)
        if m:
            assert h[want[int(m.group(1))]] > 0, (fn, dict(h))

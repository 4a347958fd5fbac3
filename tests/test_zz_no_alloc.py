"""sbf_query_seq_static: the sequence query for callers that are not allowed to allocate device memory.

Why it exists: the handle-based calls cudaMalloc their working memory (the 2-bit packed sequence and its validity
mask) and grow it on demand.  A program whose device memory was given in full to its own arena or to a framework's
caching allocator, a loop that cannot afford the device-wide synchronisation of cudaMalloc / cudaFree, or a plug-in held
to a fixed memory budget cannot let a library do that.  sbf_query_seq_static takes the filter, the sequence and the
result bitmap from the caller and keeps its working memory in one fixed array that is part of the library image
(6 MiB per GPU, hence at most 2^24 symbols per call); it calls no allocating routine at all.

What is checked: its bitmap equals the handle-based sbf_query_seq's bit for bit (this repository's bar for the query:
integer work, exact equality) — on two calls in a row that share the array, the second shorter than the first so that
the first call's leftovers lie behind it; with a filter in the caller's own memory; through the runtime-parameter
kernel; at the size limit; and that a sequence above the limit is refused with a message naming the limit.

The file is named test_zz_* so that pytest collects it last: under `pytest -x` a failure here hides no other test.
It needs nothing from the tests before it and passes alone in a fresh process as well.
"""
import numpy as np
import pytest

import seqgen
import paper_2606_24417_b200 as sbf

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

DEFAULT = dict(k=31, m=16, s=28, H=4)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def sequence(seed, n, n_runs=0):
    """Order-3 Markov DNA, optionally with runs of N (non-ACGT symbols reset the k-mer window)."""
    seq = seqgen.markov(seed, 3, 0.45, n)
    if n_runs:
        seqgen.plant_n_runs(seed + 1, seq, n_runs, 1, 40)
    return seq


def query_handle(f, d_seq):
    """The existing path: sbf_query_seq on a handle (scratch from cudaMalloc)."""
    n = d_seq.numel()
    bm = torch.full(((n + 31) // 32,), -1, dtype=torch.int32, device="cuda")  # poisoned: every word must be written
    sbf.sbf_query_seq(f.handle, d_seq, n, bm)
    torch.cuda.synchronize()
    return bm.cpu().numpy().view(np.uint32)


def query_static(params, d_filter, num_shards, d_seq, stream=None):
    """The entry point under test: no handle, the filter passed as a plain device pointer."""
    n = d_seq.numel()
    bm = torch.full(((n + 31) // 32,), -1, dtype=torch.int32, device="cuda")
    sbf.sbf_query_seq_static(params["k"], params["m"], params["s"], params["H"], d_filter, num_shards, d_seq, n, bm, stream)
    torch.cuda.synchronize()
    return bm.cpu().numpy().view(np.uint32)


def assert_same(got, want, what):
    if not np.array_equal(got, want):
        bad = np.flatnonzero(got != want)
        raise AssertionError("%s: bitmap differs in %d words of %d, first word %d: got %08x want %08x" %
                             (what, bad.size, got.size, bad[0], got[bad[0]], want[bad[0]]))


def run_pair(params, num_bits, expect_specialized):
    """Insert one sequence, then query two others (first long, then short) through both paths, in a row."""
    inserted = sequence(11, 400_000, n_runs=50)
    # half of each query is a slice of what was inserted (hits), half is foreign (misses and a few false positives)
    q_long = np.concatenate([inserted[1000:150_000], sequence(21, 150_037, n_runs=20)])   # ragged: not a multiple of 32
    q_short = np.concatenate([sequence(31, 20_011, n_runs=5), inserted[200_000:250_000]])
    with sbf.SuperBloomFilter(num_bits=num_bits, **params) as f:
        assert f.specialized == expect_specialized
        d_ins = dev(inserted)
        sbf.sbf_insert_seq(f.handle, d_ins, d_ins.numel())
        torch.cuda.synchronize()
        d_long, d_short = dev(q_long), dev(q_short)
        want_long, want_short = query_handle(f, d_long), query_handle(f, d_short)
        assert want_long.any() and want_short.any()          # the comparison is not between two empty bitmaps
        fptr, shards = sbf.sbf_filter_device_ptr(f.handle), f.num_shards
        # two calls in a row on the shared array: the short one runs over the long one's leftovers
        assert_same(query_static(params, fptr, shards, d_long), want_long, "first call")
        assert_same(query_static(params, fptr, shards, d_short), want_short, "second call (shorter, stale words behind it)")
        assert_same(query_static(params, fptr, shards, d_long), want_long, "third call (long again)")
        # a filter that lives in the caller's own memory (here: a torch tensor filled from the exported bytes)
        own = dev(f.export_bits())
        assert own.data_ptr() % 32 == 0
        assert_same(query_static(params, own, shards, d_short), want_short, "caller-owned filter")
        # on a side stream as well
        st = torch.cuda.Stream()
        torch.cuda.synchronize()
        assert_same(query_static(params, own, shards, d_long, stream=st), want_long, "side stream")


def test_static_query_matches_handle_query_specialized():
    run_pair(DEFAULT, 1 << 24, expect_specialized=True)


def test_static_query_matches_handle_query_runtime_kernel():
    """(k,m,s,H) without a compiled instance: both paths run the runtime-parameter kernel."""
    run_pair(dict(k=23, m=11, s=19, H=3), 1 << 22, expect_specialized=False)


def test_static_query_allocates_nothing_and_respects_the_limit():
    """At the limit (2^24 symbols) the result still matches; the calls leave the device's free memory unchanged;
    one symbol more is refused with a message that names the limit; an empty call is fine."""
    n_max = sbf.STATIC_MAX_SYMBOLS
    seq = sequence(41, n_max, n_runs=200)
    with sbf.SuperBloomFilter(num_bits=1 << 26, **DEFAULT) as f:
        d = dev(seq)
        sbf.sbf_insert_seq(f.handle, d[: n_max // 2], n_max // 2)
        torch.cuda.synchronize()
        want = query_handle(f, d)
        fptr, shards = sbf.sbf_filter_device_ptr(f.handle), f.num_shards
        bm = torch.full(((n_max + 31) // 32,), -1, dtype=torch.int32, device="cuda")
        args = (DEFAULT["k"], DEFAULT["m"], DEFAULT["s"], DEFAULT["H"], fptr, shards)
        sbf.sbf_query_seq_static(*args, d, 0, bm)          # empty call: does the per-device set-up, enqueues nothing
        sbf.sbf_query_seq_static(*args, d, n_max, bm)      # warm-up (first launch loads the kernels)
        torch.cuda.synchronize()
        free_before, _ = torch.cuda.mem_get_info()
        for _ in range(2):
            bm.fill_(-1)
            sbf.sbf_query_seq_static(*args, d, n_max, bm)
            torch.cuda.synchronize()
            assert_same(bm.cpu().numpy().view(np.uint32), want, "at the limit")
        free_after, _ = torch.cuda.mem_get_info()
        assert free_after == free_before, "device free memory changed by %d bytes" % (free_before - free_after)
        with pytest.raises(sbf.SBFError) as e:
            sbf.sbf_query_seq_static(*args, d, n_max + 1, bm)
        assert e.value.code == sbf.SBF_ERR_INVALID_ARG and "SBF_STATIC_MAX_SYMBOLS" in str(e.value)
        # bad geometry is refused too, before anything is enqueued
        with pytest.raises(sbf.SBFError):
            sbf.sbf_query_seq_static(31, 16, 28, 4, fptr, shards - 1, d, 64, bm)
        with pytest.raises(sbf.SBFError):
            sbf.sbf_query_seq_static(31, 16, 28, 4, fptr + 8, shards, d, 64, bm)

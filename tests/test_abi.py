"""CPU-side checks of the boundary: the C-ABI library builds, loads, and exports every symbol that
include/sbf.h declares; argument errors come back as codes; no compute call is made (no GPU here)."""
import ctypes
import os
import re

import pytest

import paper_2606_24417_b200 as sbf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols(header="sbf.h"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sbf_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported_and_bound():
    L = sbf.load_library()
    names = _declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), "libsbf_b200.so does not export %s" % n
        assert n in sbf.ABI, "python binding has no entry for %s" % n
    # and the binding binds nothing the header does not declare
    assert sorted(sbf.ABI) == names
    # same-name python wrappers exist
    for n in names:
        if n != "sbf_last_error":
            assert callable(getattr(sbf, n)), n


def test_bench_header_lives_in_its_own_library():
    """include/sbf_bench.h (ceiling micro-benchmarks, pack test hook) is exported by libsbf_bench_b200.so only: the
    product library carries none of it, and the product header declares none of it."""
    B = sbf.load_bench_library()
    L = sbf.load_library()
    names = _declared_symbols("sbf_bench.h")
    assert names == sorted(sbf.BENCH_ABI) and len(names) == 5
    for n in names:
        assert hasattr(B, n), "libsbf_bench_b200.so does not export %s" % n
        assert not hasattr(L, n), "the product library exports the bench symbol %s" % n
        assert n not in _declared_symbols("sbf.h")
        assert callable(getattr(sbf, n))
    assert not hasattr(L, "sbf_debug_last_packed")


def test_header_has_no_torch_or_cuda_types():
    text = open(os.path.join(ROOT, "include", "sbf.h")).read() + open(os.path.join(ROOT, "include", "sbf_bench.h")).read()
    code = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    assert "torch" not in code and "at::" not in code and "cuda_runtime" not in code
    assert 'extern "C"' in code


def test_invalid_arguments_fail_without_a_device():
    L = sbf.load_library()
    # bad parameters are rejected before any CUDA call
    for args in [(0, 1, 1, 1, 1024), (65, 16, 28, 4, 1024), (31, 32, 28, 4, 1024), (31, 16, 32, 4, 1024),
                 (31, 16, 28, 0, 1024), (31, 16, 28, 33, 1024), (31, 16, 28, 4, 0)]:
        assert not L.sbf_create(*args)
        assert b"sbf_create" in L.sbf_last_error()
    # k * symbol bits <= 128 (A20): protein k <= 25, DNA triplets k <= 21; unknown alphabet
    for args in [(26, 6, 20, 4, 1024, sbf.ALPHABET_PROTEIN), (22, 9, 18, 4, 1024, sbf.ALPHABET_DNA_TRIPLET), (12, 6, 10, 4, 1024, 7)]:
        assert not L.sbf_create_ex(*args)
        assert b"sbf_create" in L.sbf_last_error()
    assert L.sbf_insert_seq(None, None, 0, None) == sbf.SBF_ERR_INVALID_ARG
    assert L.sbf_query_seq(None, None, 0, None, None, None) == sbf.SBF_ERR_INVALID_ARG
    assert L.sbf_export_bits(None, None, 0) == sbf.SBF_ERR_INVALID_ARG
    assert L.sbf_num_bits(None) == 0 and L.sbf_num_shards(None) == 0
    L.sbf_destroy(None)  # ignored


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    with pytest.raises(sbf.SBFError):
        sbf.sbf_create(31, 16, 28, 4, 1 << 20)


def test_product_does_not_touch_the_oracle():
    """Nothing under the package or the C sources imports, includes or links oracle/."""
    pkg = os.path.join(ROOT, "paper_2606_24417_b200")
    for dirpath, _, files in os.walk(pkg):
        if "build" in dirpath.split(os.sep):
            continue
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                t = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in t and "from oracle" not in t and "sbf_oracle" not in t, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c", ".h")):
            t = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "paper_2606_24417_b200 import" not in t and "import paper_2606_24417_b200" not in t, fn
            assert "sbf_device" not in t and '"sbf.h"' not in t, fn

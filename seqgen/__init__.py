"""Seeded synthetic DNA workloads shared by the oracle's tests and the CUDA path.

Input generation only — none of the filter's arithmetic lives here (no packing,
hashing or filter access), so importing this module from both sides does not
couple the oracle to the CUDA path.  The C source ``seqgen.c`` is compiled on
first use into ``libseqgen.so`` beside it (gcc, OpenMP).

The five workloads follow BASELINE.json ``configs`` (recipes: DESIGN.md "Input
recipe").  They stand in for the C. elegans and T2T-CHM13 references the paper
measures on, which are not available offline.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field
from typing import Callable, Dict, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "seqgen.c")
_LIB = os.path.join(_HERE, "libseqgen.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile seqgen.c -> libseqgen.so (in-tree)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build())
    u64, u32, dbl, p = ctypes.c_uint64, ctypes.c_uint32, ctypes.c_double, ctypes.c_void_p
    lib.sg_rnd.restype = u64
    lib.sg_rnd.argtypes = [u64, u64, u64]
    lib.sg_uniform.argtypes = [u64, p, u64]
    lib.sg_markov.argtypes = [u64, ctypes.c_int, dbl, p, u64]
    lib.sg_plant_copies.argtypes = [u64, p, u64, u32, u64, u64, dbl]
    lib.sg_plant_families.argtypes = [u64, p, u64, u32, p, dbl, dbl, dbl]
    lib.sg_plant_n_runs.argtypes = [u64, p, u64, u32, u64, u64]
    lib.sg_read_start.restype = u64
    lib.sg_read_start.argtypes = [u64, u64, u32, u64]
    lib.sg_read_is_sub.restype = ctypes.c_int
    lib.sg_read_is_sub.argtypes = [u64, dbl, u32, u64, u32]
    lib.sg_reads.argtypes = [u64, p, u64, u64, u64, u32, dbl, p]
    lib.sg_record_offsets.argtypes = [u64, u64, u32, u64, u64, p]
    lib.sg_num_threads.restype = ctypes.c_int
    _lib = lib
    return lib


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def rnd(seed: int, stream: int, index: int) -> int:
    return int(_load().sg_rnd(seed, stream, index))


def uniform(seed: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.uint8)
    _load().sg_uniform(seed, _ptr(out), n)
    return out


def markov(seed: int, order: int, gc: float, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.uint8)
    _load().sg_markov(seed, order, gc, _ptr(out), n)
    return out


def plant_copies(seed, seq, n_rep, len_lo, len_hi, div):
    _load().sg_plant_copies(seed, _ptr(seq), seq.size, n_rep, len_lo, len_hi, div)


def plant_families(seed, seq, fam_len, frac, div_lo, div_hi):
    fl = np.asarray(fam_len, dtype=np.uint64)
    _load().sg_plant_families(seed, _ptr(seq), seq.size, fl.size, _ptr(fl), frac, div_lo, div_hi)


def plant_n_runs(seed, seq, n_runs, len_lo, len_hi):
    _load().sg_plant_n_runs(seed, _ptr(seq), seq.size, n_runs, len_lo, len_hi)


def reads(seed, seq, first, n_reads, read_len, sub_rate, out: Optional[np.ndarray] = None) -> np.ndarray:
    """Reads [first, first+n_reads): even index sampled from seq with substitutions, odd uniform."""
    if out is None:
        out = np.empty(n_reads * read_len, dtype=np.uint8)
    assert out.size >= n_reads * read_len and out.dtype == np.uint8
    _load().sg_reads(seed, _ptr(seq), 0 if seq is None else seq.size, first, n_reads, read_len, sub_rate, _ptr(out))
    return out


def read_start(seed, n, read_len, r) -> int:
    return int(_load().sg_read_start(seed, n, read_len, r))


def read_is_sub(seed, sub_rate, read_len, r, i) -> bool:
    return bool(_load().sg_read_is_sub(seed, sub_rate, read_len, r, i))


def record_offsets(seed, total, n_rec, lo, hi) -> np.ndarray:
    off = np.empty(n_rec + 1, dtype=np.uint64)
    _load().sg_record_offsets(seed, total, n_rec, lo, hi, _ptr(off))
    return off


def num_threads() -> int:
    return int(_load().sg_num_threads())


# ---- device-side generator (seqgen_cuda.cu): the uniform stream produced on the GPU -------------------------
_CU_SRC = os.path.join(_HERE, "seqgen_cuda.cu")
_CU_LIB = os.path.join(_HERE, "libseqgen_cuda.so")
_cu_lib = None


def build_cuda(force: bool = False) -> str:
    """Compile seqgen_cuda.cu -> libseqgen_cuda.so for sm_100a (nvcc cross-compiles without a GPU)."""
    if force or not os.path.exists(_CU_LIB) or os.path.getmtime(_CU_LIB) < os.path.getmtime(_CU_SRC):
        nvcc = "/usr/local/cuda/bin/nvcc" if os.path.exists("/usr/local/cuda/bin/nvcc") else "nvcc"
        tmp = _CU_LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-shared",
                               "-Xcompiler", "-fPIC", "-o", tmp, _CU_SRC])
        os.replace(tmp, _CU_LIB)
    return _CU_LIB


def uniform_device(seed: int, first: int, n: int, out=None, stream=None):
    """Symbols [first, first + n) of the uniform(seed, .) stream as a CUDA uint8 tensor, generated on the device
    (byte-identical to uniform(seed, first + n)[first:])."""
    import torch
    global _cu_lib
    if _cu_lib is None:
        _cu_lib = ctypes.CDLL(build_cuda())
        _cu_lib.sg_uniform_device.restype = ctypes.c_int
        _cu_lib.sg_uniform_device.argtypes = [ctypes.c_uint64, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint64,
                                              ctypes.c_void_p]
    if out is None:
        out = torch.empty(n, dtype=torch.uint8, device="cuda")
    assert out.is_cuda and out.dtype == torch.uint8 and out.numel() >= n and out.is_contiguous()
    st = None if stream is None else stream.cuda_stream
    rc = _cu_lib.sg_uniform_device(seed, out.data_ptr(), first, n, st)
    if rc != 0:
        raise RuntimeError("sg_uniform_device: CUDA error %d" % rc)
    return out


def fasta_text(records, width: int = 60, crlf: bool = False, names=None) -> bytes:
    """FASTA text of the given records (uint8 arrays / bytes): '>name' line, then the sequence wrapped at `width`."""
    eol = b"\r\n" if crlf else b"\n"
    out = bytearray()
    for i, r in enumerate(records):
        b = bytes(r)
        out += b">" + (names[i] if names else b"rec%d some description" % i) + eol
        for a in range(0, len(b), width):
            out += b[a:a + width] + eol
    return bytes(out)


def fastq_text(records, crlf: bool = False, final_newline: bool = True) -> bytes:
    """Four-line FASTQ text of the given records; the quality line is a seeded pattern that contains '>' and '@'."""
    eol = b"\r\n" if crlf else b"\n"
    qual = b"IIII>@FF#5;"
    out = bytearray()
    for i, r in enumerate(records):
        b = bytes(r)
        q = (qual * (len(b) // len(qual) + 1))[:len(b)]
        out += b"@read%d/1" % i + eol + b + eol + b"+" + eol + q + eol
    if not final_newline and out.endswith(eol):
        del out[-len(eol):]
    return bytes(out)


def fixed_offsets(n_reads: int, read_len: int, first: int = 0) -> np.ndarray:
    """offsets[n_reads+1] of back-to-back fixed-length records (relative to the batch)."""
    return (np.arange(n_reads + 1, dtype=np.uint64) * np.uint64(read_len))


# ----------------------------------------------------------------------------
# The five BASELINE.json configs.  `scale` < 1 shrinks base and read counts for
# CPU-sized tests (filter size is scaled by the caller if it wants to).
# ----------------------------------------------------------------------------

DEFAULT_PARAMS = dict(k=31, m=16, s=28, H=4)


@dataclass
class Workload:
    name: str
    params: Dict[str, int]               # k, m, s, H, num_bits
    insert_bases: np.ndarray             # uint8 ASCII, all records concatenated
    insert_offsets: np.ndarray           # uint64[n_rec+1]
    n_reads: int = 0
    read_len: int = 150
    read_sub_rate: float = 0.01
    read_seed: int = 0
    extra: Dict[str, object] = field(default_factory=dict)

    def read_batch(self, first: int, count: int, out: Optional[np.ndarray] = None) -> np.ndarray:
        return reads(self.read_seed, self.insert_bases, first, count, self.read_len, self.read_sub_rate, out)


def config1() -> Workload:
    """Tiny: 1 Mbp uniform (seed 1), filter 2^20 bits; aliens = 1 Mbp uniform (seed 2)."""
    seq = uniform(1, 1_000_000)
    w = Workload("config1-tiny", dict(DEFAULT_PARAMS, num_bits=1 << 20), seq,
                 np.array([0, seq.size], dtype=np.uint64))
    w.extra["alien"] = uniform(2, 1_000_000)
    return w


def config2(scale: float = 1.0, n_reads: Optional[int] = None) -> Workload:
    """Bacterial-scale: 5 Mbp order-3 Markov (GC 50%), 200 copied repeats of 1-5 kb at 0.5%."""
    n = max(20_000, int(5_000_000 * scale))
    seq = markov(21, 3, 0.50, n)
    plant_copies(22, seq, max(1, int(200 * scale)), 1000, 5000, 0.005)
    w = Workload("config2-bacterial", dict(DEFAULT_PARAMS, num_bits=0), seq,
                 np.array([0, n], dtype=np.uint64),
                 n_reads=int(1_000_000 * scale) if n_reads is None else n_reads, read_seed=23)
    return w


def count_distinct_windows(seq: np.ndarray, k: int) -> int:
    """Exact number of distinct length-k substrings made of ACGT only (plain string set)."""
    s = seq.tobytes()
    bad = set(range(256)) - set(b"ACGTacgt")
    table = bytes(1 if c in bad else 0 for c in range(256))
    flags = np.frombuffer(s.translate(table), dtype=np.uint8)
    csum = np.concatenate(([0], np.cumsum(flags, dtype=np.int64)))
    ok = (csum[k:] - csum[:-k]) == 0
    up = s.upper()
    return len({up[i:i + k] for i in np.flatnonzero(ok)})


def config3(scale: float = 1.0, n_reads: Optional[int] = None) -> Workload:
    """Chromosome-scale: 250 Mbp order-5 Markov (GC 41%), 100 N runs of 10-50 kb, filter 2^32 bits."""
    n = max(100_000, int(250_000_000 * scale))
    seq = markov(31, 5, 0.41, n)
    plant_n_runs(32, seq, max(1, int(round(100 * scale))), 10_000, 50_000)
    w = Workload("config3-chromosome", dict(DEFAULT_PARAMS, num_bits=1 << 32), seq,
                 np.array([0, n], dtype=np.uint64),
                 n_reads=int(40_000_000 * scale) if n_reads is None else n_reads, read_seed=33)
    return w


def config4(scale: float = 1.0, n_reads: Optional[int] = None) -> Workload:
    """Genome-scale: 3.1 Gbp in 24 records (50-250 Mbp), ~5% repeat families, filter 2^35 bits."""
    n = max(1_000_000, int(3_100_000_000 * scale))
    off = record_offsets(44, n, 24, 50_000_000, 250_000_000)
    seq = markov(41, 5, 0.41, n)
    plant_families(42, seq, [300] * 6 + [6000] * 2, 0.05, 0.10, 0.20)
    w = Workload("config4-genome", dict(DEFAULT_PARAMS, num_bits=1 << 35), seq, off,
                 n_reads=int(100_000_000 * scale) if n_reads is None else n_reads, read_seed=43)
    return w


SWEEP_S = (24, 26, 28, 30, 31)
SWEEP_M = (12, 14, 16, 18, 20)
SWEEP_H = (1, 2, 4, 6, 8)
SWEEP_LOG2_BITS = tuple(range(28, 35))


def config5_points(full_cross: bool = True):
    """(s, m, H) points of the sweep: the 125-point cross product or the three axes through (28,16,4)."""
    if full_cross:
        return [(s, m, h) for s in SWEEP_S for m in SWEEP_M for h in SWEEP_H]
    pts = {(s, 16, 4) for s in SWEEP_S} | {(28, m, 4) for m in SWEEP_M} | {(28, 16, h) for h in SWEEP_H}
    return sorted(pts)

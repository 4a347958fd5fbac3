"""ctypes front end of the CPU oracle (oracle/sbf_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this.  It shares no
code with paper_2606_24417_b200 and never imports it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sbf_oracle.c")
_HDR = os.path.join(_HERE, "sbf_oracle.h")
_LIB = os.path.join(_HERE, "libsbf_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = ctypes.CDLL(build())
    u64, u32, i32, p = ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int, ctypes.c_void_p
    L.sbfo_code.restype = i32; L.sbfo_code.argtypes = [ctypes.c_ubyte]
    L.sbfo_sub.restype = u64; L.sbfo_sub.argtypes = [u64, i32, i32, i32]
    L.sbfo_g.restype = u32; L.sbfo_g.argtypes = [i32, u64]
    L.sbfo_sigma.restype = u64; L.sbfo_sigma.argtypes = [u32, i32]
    L.sbfo_f.restype = u64; L.sbfo_f.argtypes = [i32, u64]
    L.sbfo_bitpos.restype = i32; L.sbfo_bitpos.argtypes = [u64, i32, i32]
    L.sbfo_create.restype = p; L.sbfo_create.argtypes = [i32, i32, i32, i32, u64]
    L.sbfo_destroy.argtypes = [p]
    L.sbfo_clear.argtypes = [p]
    L.sbfo_num_shards.restype = u64; L.sbfo_num_shards.argtypes = [p]
    L.sbfo_words.restype = p; L.sbfo_words.argtypes = [p]
    L.sbfo_pack_kmer.restype = i32; L.sbfo_pack_kmer.argtypes = [p, p, u64, u64, ctypes.POINTER(u64)]
    L.sbfo_min_key.restype = u32; L.sbfo_min_key.argtypes = [p, u64]
    L.sbfo_shard_of.restype = u64; L.sbfo_shard_of.argtypes = [p, u64]
    L.sbfo_insert_kmer.argtypes = [p, u64]
    L.sbfo_contains_kmer.restype = i32; L.sbfo_contains_kmer.argtypes = [p, u64]
    for name in ("sbfo_insert_records", "sbfo_insert_records_mt", "sbfo_count_valid_kmers"):
        fn = getattr(L, name); fn.restype = u64; fn.argtypes = [p, p, p, u64]
    for name in ("sbfo_query_records", "sbfo_query_records_mt"):
        fn = getattr(L, name); fn.restype = u64; fn.argtypes = [p, p, p, u64, p, p]
    L.sbfo_trace_records.restype = u64; L.sbfo_trace_records.argtypes = [p, p, p, u64, p, p, p]
    L.sbfo_num_threads.restype = i32
    # wide path (A19-A22)
    L.sbfo_create_ex.restype = p; L.sbfo_create_ex.argtypes = [i32, i32, i32, i32, u64, i32]
    L.sbfo_force_wide.argtypes = [p, i32]
    L.sbfo_symbol_code.restype = i32; L.sbfo_symbol_code.argtypes = [i32, p]
    L.sbfo_fold64.restype = u64; L.sbfo_fold64.argtypes = [u64, u64]
    L.sbfo_pack_kmer_w.restype = i32; L.sbfo_pack_kmer_w.argtypes = [p, p, u64, u64, ctypes.POINTER(u64), ctypes.POINTER(u64)]
    L.sbfo_sub_w.restype = u64; L.sbfo_sub_w.argtypes = [p, u64, u64, i32, i32]
    L.sbfo_min_key_w.restype = u32; L.sbfo_min_key_w.argtypes = [p, u64, u64]
    L.sbfo_shard_of_w.restype = u64; L.sbfo_shard_of_w.argtypes = [p, u64, u64]
    L.sbfo_insert_kmer_w.argtypes = [p, u64, u64]
    L.sbfo_contains_kmer_w.restype = i32; L.sbfo_contains_kmer_w.argtypes = [p, u64, u64]
    _lib = L
    return L


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _as_bases(x) -> np.ndarray:
    if isinstance(x, (bytes, bytearray, str)):
        x = np.frombuffer(x.encode() if isinstance(x, str) else bytes(x), dtype=np.uint8)
    return np.ascontiguousarray(x, dtype=np.uint8)


def _as_offsets(offsets, total) -> np.ndarray:
    if offsets is None:
        return np.array([0, total], dtype=np.uint64)
    return np.ascontiguousarray(offsets, dtype=np.uint64)


class OracleSBF:
    """The oracle's filter object; mirrors the C-ABI names of the product for readability only."""

    def __init__(self, k: int, m: int, s: int, H: int, num_bits: int, alphabet: int = 0):
        self._L = lib()
        self._h = (self._L.sbfo_create(k, m, s, H, num_bits) if alphabet == 0 and k <= 32 else
                   self._L.sbfo_create_ex(k, m, s, H, num_bits, alphabet))
        if not self._h:
            raise ValueError("oracle: invalid parameters k=%d m=%d s=%d H=%d num_bits=%d alphabet=%d" % (k, m, s, H, num_bits, alphabet))
        self.k, self.m, self.s, self.H, self.alphabet = k, m, s, H, alphabet
        self.num_shards = int(self._L.sbfo_num_shards(self._h))

    def close(self):
        if self._h:
            self._L.sbfo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def num_bits(self) -> int:
        return self.num_shards * 256

    def clear(self):
        self._L.sbfo_clear(self._h)

    def words(self) -> np.ndarray:
        """View of the filter as uint64[num_shards, 4] (A12 layout)."""
        n = self.num_shards * 4
        buf = (ctypes.c_uint64 * n).from_address(self._L.sbfo_words(self._h))
        return np.frombuffer(buf, dtype=np.uint64).reshape(self.num_shards, 4)

    def export_bits(self) -> np.ndarray:
        return self.words().reshape(-1).view(np.uint8).copy()

    # ---- batches ----
    def insert_records(self, bases, offsets=None, threads: bool = False) -> int:
        b = _as_bases(bases); o = _as_offsets(offsets, b.size)
        fn = self._L.sbfo_insert_records_mt if threads else self._L.sbfo_insert_records
        return int(fn(self._h, _ptr(b), _ptr(o), o.size - 1))

    insert_seq = insert_records

    def query_records(self, bases, offsets=None, want_counts: bool = True, threads: bool = False):
        b = _as_bases(bases); o = _as_offsets(offsets, b.size)
        bitmap = np.zeros((b.size + 31) // 32, dtype=np.uint32)
        counts = np.zeros(o.size - 1, dtype=np.uint32) if want_counts else None
        fn = self._L.sbfo_query_records_mt if threads else self._L.sbfo_query_records
        nv = int(fn(self._h, _ptr(b), _ptr(o), o.size - 1, _ptr(bitmap), _ptr(counts)))
        return bitmap, counts, nv

    query_seq = query_records

    def count_valid_kmers(self, bases, offsets=None) -> int:
        b = _as_bases(bases); o = _as_offsets(offsets, b.size)
        return int(self._L.sbfo_count_valid_kmers(self._h, _ptr(b), _ptr(o), o.size - 1))

    def trace(self, bases, offsets=None):
        """(min_key uint32[n], shard uint64[n], valid bool[n]) per global base position."""
        b = _as_bases(bases); o = _as_offsets(offsets, b.size)
        mk = np.zeros(b.size, dtype=np.uint32); sh = np.zeros(b.size, dtype=np.uint64)
        va = np.zeros(b.size, dtype=np.uint8)
        self._L.sbfo_trace_records(self._h, _ptr(b), _ptr(o), o.size - 1, _ptr(mk), _ptr(sh), _ptr(va))
        return mk, sh, va.astype(bool)

    # ---- single k-mers ----
    def pack_kmer(self, rec, p: int):
        b = _as_bases(rec); v = ctypes.c_uint64(0)
        ok = self._L.sbfo_pack_kmer(self._h, _ptr(b), b.size, p, ctypes.byref(v))
        return (int(v.value) if ok else None)

    def min_key(self, v: int) -> int:
        return int(self._L.sbfo_min_key(self._h, v))

    def shard_of(self, v: int) -> int:
        return int(self._L.sbfo_shard_of(self._h, v))

    def insert_kmer(self, v: int):
        self._L.sbfo_insert_kmer(self._h, v)

    def contains_kmer(self, v: int) -> bool:
        return bool(self._L.sbfo_contains_kmer(self._h, v))

    # ---- wide path: a packed k-mer is a Python int below 2^128 ----
    def force_wide(self, on: bool = True):
        self._L.sbfo_force_wide(self._h, 1 if on else 0)

    def pack_kmer_w(self, rec, p: int):
        b = _as_bases(rec); hi, lo = ctypes.c_uint64(0), ctypes.c_uint64(0)
        ok = self._L.sbfo_pack_kmer_w(self._h, _ptr(b), b.size, p, ctypes.byref(hi), ctypes.byref(lo))
        return ((int(hi.value) << 64) | int(lo.value)) if ok else None

    def sub_w(self, v: int, i: int, ln: int) -> int:
        return int(self._L.sbfo_sub_w(self._h, v >> 64, v & _M64, i, ln))

    def min_key_w(self, v: int) -> int:
        return int(self._L.sbfo_min_key_w(self._h, v >> 64, v & _M64))

    def shard_of_w(self, v: int) -> int:
        return int(self._L.sbfo_shard_of_w(self._h, v >> 64, v & _M64))

    def insert_kmer_w(self, v: int):
        self._L.sbfo_insert_kmer_w(self._h, v >> 64, v & _M64)

    def contains_kmer_w(self, v: int) -> bool:
        return bool(self._L.sbfo_contains_kmer_w(self._h, v >> 64, v & _M64))


_M64 = (1 << 64) - 1
DNA, PROTEIN, TRIPLET = 0, 1, 2


def fold64(hi, lo): return int(lib().sbfo_fold64(hi, lo))


def symbol_code(alphabet, sym: bytes) -> int:
    b = np.frombuffer(bytes(sym) + b"\0\0", dtype=np.uint8).copy()
    return int(lib().sbfo_symbol_code(alphabet, _ptr(b)))


def g(m, x): return int(lib().sbfo_g(m, x))
def sigma(key, P): return int(lib().sbfo_sigma(key, P))
def f(s, x): return int(lib().sbfo_f(s, x))
def bitpos(h, i, H): return int(lib().sbfo_bitpos(h, i, H))
def sub(v, k, i, ln): return int(lib().sbfo_sub(v, k, i, ln))
def code(c): return int(lib().sbfo_code(c if isinstance(c, int) else ord(c)))
def num_threads(): return int(lib().sbfo_num_threads())


def bitmap_bits(bitmap: np.ndarray, n: int) -> np.ndarray:
    """uint32 bitmap -> bool[n] (bit p = word p>>5, bit p&31)."""
    return np.unpackbits(bitmap.view(np.uint8), bitorder="little")[:n].astype(bool)

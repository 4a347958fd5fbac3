"""paper_2606_24417_b200 — B200-native Super Bloom filter insert/query hot path (arxiv 2606.24417).

Thin ctypes binding over the C ABI of ``include/sbf.h`` (``libsbf_b200.so``, hand-written CUDA for
sm_100a).  The functions below have the C names and do argument marshalling only; every step of
the path runs in the library's kernels.  There is no CPU fallback: if the library is missing or no
CUDA device is present the calls raise.

PyTorch is used by callers for device buffers and streams only; this module accepts raw device
pointers (ints), ``torch`` CUDA tensors, or for the ``*_host`` calls numpy arrays / pinned tensors.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsbf_b200.so")
BENCH_LIB_PATH = os.path.join(_HERE, "libsbf_bench_b200.so")
_lib = None
_bench_lib = None

SBF_OK = 0
SBF_ERR_INVALID_ARG = -1
SBF_ERR_UNSUPPORTED = -2
SBF_ERR_NOMEM = -3
SBF_ERR_CUDA = -4

# every symbol include/sbf.h declares: name -> (restype, argtypes)
_u64, _u32, _i32, _p, _cp = ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int, ctypes.c_void_p, ctypes.c_char_p
ABI = {
    "sbf_create": (_p, [_i32, _i32, _i32, _i32, _u64]),
    "sbf_create_ex": (_p, [_i32, _i32, _i32, _i32, _u64, _i32]),
    "sbf_destroy": (None, [_p]),
    "sbf_num_bits": (_u64, [_p]),
    "sbf_num_shards": (_u64, [_p]),
    "sbf_is_specialized": (_i32, [_p]),
    "sbf_reserve": (_i32, [_p, _u64]),
    "sbf_clear": (_i32, [_p, _p]),
    "sbf_insert_seq": (_i32, [_p, _p, _u64, _p]),
    "sbf_insert_records": (_i32, [_p, _p, _p, _u64, _u64, _p]),
    "sbf_query_seq": (_i32, [_p, _p, _u64, _p, _p, _p]),
    "sbf_query_records": (_i32, [_p, _p, _p, _u64, _u64, _p, _p, _p]),
    "sbf_query_seq_static": (_i32, [_i32, _i32, _i32, _i32, _p, _u64, _p, _u64, _p, _p]),
    "sbf_insert_seq_host": (_i32, [_p, _p, _u64]),
    "sbf_insert_records_host": (_i32, [_p, _p, _p, _u64]),
    "sbf_query_seq_host": (_i32, [_p, _p, _u64, _p, _p]),
    "sbf_query_records_host": (_i32, [_p, _p, _p, _u64, _p, _p]),
    "sbf_insert_fastx_host": (_i32, [_p, _p, _u64, _i32, _p, _p]),
    "sbf_query_fastx_host": (_i32, [_p, _p, _u64, _i32, _p, _u64, _p, _p]),
    "sbf_export_bits": (_i32, [_p, _p, _u64]),
    "sbf_import_bits": (_i32, [_p, _p, _u64]),
    "sbf_filter_device_ptr": (_p, [_p]),
    "sbf_or_bits_device": (_i32, [_p, _p, _u64, _p]),
    "sbf_or_range_device": (_i32, [_p, _u64, _p, _u64, _p]),
    "sbf_or_peers_range_device": (_i32, [_p, _u64, _p, _i32, _u64, _p]),
    "sbf_ipc_export_filter": (_i32, [_p, _p]),
    "sbf_ipc_open_filter": (_i32, [_p, _p]),
    "sbf_ipc_close_filter": (_i32, [_p]),
    "sbf_last_error": (_cp, []),
    "sbf_kernel_launches": (_u64, []),
    "sbf_set_host_chunk": (_i32, [_p, _u64]),
    "sbf_set_timing": (_i32, [_p, _i32]),
    "sbf_get_timing": (_i32, [_p, _p]),
}
# every symbol include/sbf_bench.h declares (libsbf_bench_b200.so: measurement and test hooks, not the product boundary)
BENCH_ABI = {
    "sbf_ceiling_pipe_modes": (_i32, []),
    "sbf_ceiling_pipe_mode_name": (_cp, [_i32]),
    "sbf_ceiling_pipe_rate": (_i32, [_i32, _i32, _p, _p]),
    "sbf_ceiling_random_sector": (_i32, [_i32, _u64, _p]),
    "sbf_bench_pack": (_i32, [_p, _u64, _i32, _p, _p, _u64]),
}


class SBFError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__("sbf error %d: %s" % (code, msg))
        self.code = code


def load_library(build_if_missing: bool = True):
    """dlopen libsbf_b200.so and type every symbol.  With build_if_missing the (mtime-incremental) build runs
    first, so a library older than its sources is never loaded; without nvcc an existing library is used as is."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing and LIB_PATH == os.path.join(_HERE, "libsbf_b200.so"):
        from . import build as _build
        try:
            _build.build()
        except FileNotFoundError:          # no nvcc on this box: fall through to whatever was shipped
            pass
    if not os.path.exists(LIB_PATH):
        raise SBFError(SBF_ERR_UNSUPPORTED, "libsbf_b200.so not built (python -m paper_2606_24417_b200.build)")
    L = ctypes.CDLL(LIB_PATH)
    for name, (res, args) in ABI.items():
        fn = getattr(L, name)  # AttributeError here = the library does not export what sbf.h declares
        fn.restype = res
        fn.argtypes = args
    _lib = L
    return L


def load_bench_library():
    """dlopen libsbf_bench_b200.so (include/sbf_bench.h) — bench.py, the ceilings CLI and the tests only."""
    global _bench_lib
    if _bench_lib is not None:
        return _bench_lib
    load_library()                          # runs the incremental build of both libraries
    if not os.path.exists(BENCH_LIB_PATH):
        raise SBFError(SBF_ERR_UNSUPPORTED, "libsbf_bench_b200.so not built (python -m paper_2606_24417_b200.build)")
    L = ctypes.CDLL(BENCH_LIB_PATH)
    for name, (res, args) in BENCH_ABI.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    _bench_lib = L
    return L


def _check_bench(rc: int, what: str):
    if rc != SBF_OK:
        raise SBFError(rc, "%s failed (libsbf_bench_b200.so returns codes only)" % what)


def _check(rc: int):
    if rc != SBF_OK:
        raise SBFError(rc, load_library().sbf_last_error().decode())


def _dptr(x) -> Optional[int]:
    """Device pointer of a torch CUDA tensor, or an int / None passed through."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "is_cuda"):
        if not x.is_cuda:
            raise TypeError("expected a CUDA tensor")
        if not x.is_contiguous():
            raise TypeError("expected a contiguous tensor")
        return x.data_ptr()
    raise TypeError("expected a CUDA tensor or a raw device pointer, got %r" % type(x))


def _hptr(x) -> Optional[int]:
    """Host pointer of a numpy array / CPU tensor / bytes."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, bytes):   # the caller keeps the object alive for the duration of the call
        return ctypes.cast(ctypes.c_char_p(x), ctypes.c_void_p).value
    if isinstance(x, np.ndarray):
        if not x.flags["C_CONTIGUOUS"]:
            raise TypeError("expected a C-contiguous array")
        return x.ctypes.data
    if hasattr(x, "is_cuda"):
        if x.is_cuda:
            raise TypeError("expected a host tensor")
        return x.data_ptr()
    raise TypeError("expected a numpy array, a CPU tensor or a raw host pointer, got %r" % type(x))


def _stream(stream) -> Optional[int]:
    if stream is None:
        return None
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream  # torch.cuda.Stream


# ---- the C ABI, same names -------------------------------------------------------------------
def sbf_create(k: int, m: int, s: int, H: int, num_bits: int) -> int:
    L = load_library()
    h = L.sbf_create(k, m, s, H, num_bits)
    if not h:
        raise SBFError(SBF_ERR_INVALID_ARG, L.sbf_last_error().decode())
    return h


ALPHABET_DNA, ALPHABET_PROTEIN, ALPHABET_DNA_TRIPLET = 0, 1, 2


def sbf_create_ex(k: int, m: int, s: int, H: int, num_bits: int, alphabet: int) -> int:
    L = load_library()
    h = L.sbf_create_ex(k, m, s, H, num_bits, alphabet)
    if not h:
        raise SBFError(SBF_ERR_INVALID_ARG, L.sbf_last_error().decode())
    return h


def sbf_destroy(h): load_library().sbf_destroy(h)
def sbf_num_bits(h) -> int: return int(load_library().sbf_num_bits(h))
def sbf_num_shards(h) -> int: return int(load_library().sbf_num_shards(h))
def sbf_is_specialized(h) -> bool: return bool(load_library().sbf_is_specialized(h))
def sbf_reserve(h, max_bases: int): _check(load_library().sbf_reserve(h, max_bases))
def sbf_clear(h, stream=None): _check(load_library().sbf_clear(h, _stream(stream)))
def sbf_kernel_launches() -> int: return int(load_library().sbf_kernel_launches())
def sbf_filter_device_ptr(h) -> int: return int(load_library().sbf_filter_device_ptr(h) or 0)


def sbf_insert_seq(h, d_seq, length: int, stream=None):
    _check(load_library().sbf_insert_seq(h, _dptr(d_seq), length, _stream(stream)))


def sbf_insert_records(h, d_bases, d_offsets, n_rec: int, total_bases: int, stream=None):
    _check(load_library().sbf_insert_records(h, _dptr(d_bases), _dptr(d_offsets), n_rec, total_bases, _stream(stream)))


def sbf_query_seq(h, d_seq, length: int, d_bitmap, d_hits=None, stream=None):
    _check(load_library().sbf_query_seq(h, _dptr(d_seq), length, _dptr(d_bitmap), _dptr(d_hits), _stream(stream)))


def sbf_query_records(h, d_bases, d_offsets, n_rec: int, total_bases: int, d_bitmap, d_hit_counts=None, stream=None):
    _check(load_library().sbf_query_records(h, _dptr(d_bases), _dptr(d_offsets), n_rec, total_bases, _dptr(d_bitmap),
                                            _dptr(d_hit_counts), _stream(stream)))


STATIC_MAX_SYMBOLS = 1 << 24  # SBF_STATIC_MAX_SYMBOLS of include/sbf.h


def sbf_query_seq_static(k: int, m: int, s: int, H: int, d_filter, num_shards: int, d_seq, length: int, d_bitmap, stream=None):
    """sbf_query_seq without a handle and without any device allocation, for callers that may not allocate (a process
    whose device memory belongs to its own pool, a loop that cannot take cudaMalloc's synchronisation): the working
    memory is one fixed array inside the library, shared by every call, so at most STATIC_MAX_SYMBOLS symbols per call
    and never two calls in flight at once on one GPU.  d_filter: the caller's filter (layout A12, num_shards x 32 bytes).
    See include/sbf.h."""
    _check(load_library().sbf_query_seq_static(k, m, s, H, _dptr(d_filter), num_shards, _dptr(d_seq), length,
                                               _dptr(d_bitmap), _stream(stream)))


def sbf_insert_seq_host(h, h_seq, length: int):
    _check(load_library().sbf_insert_seq_host(h, _hptr(h_seq), length))


def sbf_insert_records_host(h, h_bases, h_offsets, n_rec: int):
    _check(load_library().sbf_insert_records_host(h, _hptr(h_bases), _hptr(h_offsets), n_rec))


def sbf_query_seq_host(h, h_seq, length: int, h_bitmap, h_hits=None):
    _check(load_library().sbf_query_seq_host(h, _hptr(h_seq), length, _hptr(h_bitmap), _hptr(h_hits)))


def sbf_query_records_host(h, h_bases, h_offsets, n_rec: int, h_bitmap, h_hit_counts=None):
    _check(load_library().sbf_query_records_host(h, _hptr(h_bases), _hptr(h_offsets), n_rec, _hptr(h_bitmap),
                                                 _hptr(h_hit_counts)))


def sbf_insert_fastx_host(h, h_text, n_bytes: int, fmt: int = 0):
    """(records, sequence bytes) found in the FASTA/FASTQ text and inserted."""
    nr, nb = ctypes.c_uint64(0), ctypes.c_uint64(0)
    _check(load_library().sbf_insert_fastx_host(h, _hptr(h_text), n_bytes, fmt, ctypes.addressof(nr), ctypes.addressof(nb)))
    return int(nr.value), int(nb.value)


def sbf_query_fastx_host(h, h_text, n_bytes: int, h_hit_counts, max_records: int, fmt: int = 0):
    """Fills h_hit_counts[0 .. records); returns (records, sequence bytes)."""
    nr, nb = ctypes.c_uint64(0), ctypes.c_uint64(0)
    _check(load_library().sbf_query_fastx_host(h, _hptr(h_text), n_bytes, fmt, _hptr(h_hit_counts), max_records,
                                               ctypes.addressof(nr), ctypes.addressof(nb)))
    return int(nr.value), int(nb.value)


def sbf_export_bits(h) -> np.ndarray:
    """The filter as uint8[32*numShards] (layout A12)."""
    n = sbf_num_shards(h) * 32
    out = np.empty(n, dtype=np.uint8)
    _check(load_library().sbf_export_bits(h, out.ctypes.data, n))
    return out


def sbf_import_bits(h, bits: np.ndarray):
    b = np.ascontiguousarray(bits, dtype=np.uint8)
    _check(load_library().sbf_import_bits(h, b.ctypes.data, b.size))


def sbf_or_bits_device(h, d_src, nbytes: int, stream=None):
    _check(load_library().sbf_or_bits_device(h, _dptr(d_src), nbytes, _stream(stream)))


def sbf_or_range_device(h, offset_bytes: int, d_src, nbytes: int, stream=None):
    _check(load_library().sbf_or_range_device(h, offset_bytes, _dptr(d_src), nbytes, _stream(stream)))


def sbf_or_peers_range_device(h, offset_bytes: int, peer_range_ptrs, nbytes: int, stream=None):
    """peer_range_ptrs: raw device pointers (ints) to the start of the same range in every peer replica."""
    arr = (ctypes.c_uint64 * max(1, len(peer_range_ptrs)))(*peer_range_ptrs)
    _check(load_library().sbf_or_peers_range_device(h, offset_bytes, ctypes.addressof(arr), len(peer_range_ptrs), nbytes,
                                                    _stream(stream)))


def sbf_ipc_export_filter(h) -> bytes:
    buf = ctypes.create_string_buffer(64)
    _check(load_library().sbf_ipc_export_filter(h, ctypes.addressof(buf)))
    return buf.raw


def sbf_ipc_open_filter(handle64: bytes) -> int:
    buf = ctypes.create_string_buffer(handle64, 64)
    out = ctypes.c_uint64(0)
    _check(load_library().sbf_ipc_open_filter(ctypes.addressof(buf), ctypes.addressof(out)))
    return int(out.value)


def sbf_ipc_close_filter(ptr: int):
    _check(load_library().sbf_ipc_close_filter(ptr))


def sbf_set_host_chunk(h, symbols: int):
    _check(load_library().sbf_set_host_chunk(h, symbols))


def sbf_set_timing(h, on: bool):
    _check(load_library().sbf_set_timing(h, 1 if on else 0))


def sbf_get_timing(h):
    """(pack_ms, main_ms, count_ms) of the last device-facing call."""
    ms = (ctypes.c_float * 3)()
    _check(load_library().sbf_get_timing(h, ctypes.cast(ms, ctypes.c_void_p)))
    return float(ms[0]), float(ms[1]), float(ms[2])


def sbf_ceiling_pipe_modes() -> int: return int(load_bench_library().sbf_ceiling_pipe_modes())
def sbf_ceiling_pipe_mode_name(mode: int) -> str: return load_bench_library().sbf_ceiling_pipe_mode_name(mode).decode()


def sbf_ceiling_pipe_rate(mode: int, iters: int = 2048):
    """(1e9 warp instructions per second per SM sub-partition, clock64() rate in MHz) of one instruction mix."""
    r, c = ctypes.c_double(0), ctypes.c_double(0)
    _check_bench(load_bench_library().sbf_ceiling_pipe_rate(mode, iters, ctypes.addressof(r), ctypes.addressof(c)), "sbf_ceiling_pipe_rate")
    return float(r.value), float(c.value)


def sbf_ceiling_random_sector(mode: int, array_bytes: int) -> float:
    """Random 32-byte-sector accesses per second (1e9/s) over array_bytes."""
    g = ctypes.c_double(0)
    _check_bench(load_bench_library().sbf_ceiling_random_sector(mode, array_bytes, ctypes.addressof(g)), "sbf_ceiling_random_sector")
    return float(g.value)


def sbf_bench_pack(d_seq, length: int, k: int, n_words: int):
    """(packed 2-bit words, validity masks) of the first n_words 16-symbol words, as pack_kernel writes them."""
    w = np.empty(n_words, dtype=np.uint32)
    g = np.empty(n_words, dtype=np.uint16)
    _check_bench(load_bench_library().sbf_bench_pack(_dptr(d_seq), length, k, w.ctypes.data, g.ctypes.data, n_words), "sbf_bench_pack")
    return w, g


class SuperBloomFilter:
    """Convenience owner of one handle (context manager); methods forward to the C ABI."""

    def __init__(self, k: int = 31, m: int = 16, s: int = 28, H: int = 4, num_bits: int = 1 << 32, alphabet: int = 0):
        self.k, self.m, self.s, self.H, self.alphabet = k, m, s, H, alphabet
        self.handle = sbf_create_ex(k, m, s, H, num_bits, alphabet)
        self.num_shards = sbf_num_shards(self.handle)
        self.num_bits = sbf_num_bits(self.handle)
        self.specialized = sbf_is_specialized(self.handle)

    def close(self):
        if getattr(self, "handle", None):
            sbf_destroy(self.handle)
            self.handle = None

    def __enter__(self): return self
    def __exit__(self, *a): self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def reserve(self, max_bases): sbf_reserve(self.handle, max_bases)
    def clear(self, stream=None): sbf_clear(self.handle, stream)
    def export_bits(self): return sbf_export_bits(self.handle)
    def import_bits(self, bits): sbf_import_bits(self.handle, bits)

    def insert_seq(self, d_seq, stream=None):
        sbf_insert_seq(self.handle, d_seq, d_seq.numel(), stream)

    def insert_records(self, d_bases, d_offsets, stream=None):
        sbf_insert_records(self.handle, d_bases, d_offsets, d_offsets.numel() - 1, d_bases.numel(), stream)

    def query_seq(self, d_seq, d_bitmap, d_hits=None, stream=None):
        sbf_query_seq(self.handle, d_seq, d_seq.numel(), d_bitmap, d_hits, stream)

    def query_records(self, d_bases, d_offsets, d_bitmap, d_hit_counts=None, stream=None):
        sbf_query_records(self.handle, d_bases, d_offsets, d_offsets.numel() - 1, d_bases.numel(), d_bitmap,
                          d_hit_counts, stream)

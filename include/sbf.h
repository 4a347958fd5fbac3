/*
 * sbf.h — C ABI of the B200-native Super Bloom filter insert/query hot path.
 *
 * What the library computes is defined by the paper (arxiv 2606.24417, "cuSBF";
 * P:<n> = line n of its extracted text PAPER.md) and, where the paper gives no
 * constants or edge rules, by the readings A1-A18 in DESIGN.md §3:
 *
 *   a k-mer v (2 bits/base, first base most significant) is mapped to
 *     minKey = min over its k-m+1 m-mers of g(m-mer)             (A1)
 *     shard  = sigma(minKey) in [0, 2^P)                         (A2)
 *     for each of its k-s+1 s-mers x, h = f(x), and for i < H the bit
 *     B(h,i) of 64-bit sector word (i mod 4) of that shard       (A4, A5)
 *   insert sets those H*(k-s+1) bits (Alg. 1); query reports the k-mer
 *   present iff every one of them is set — the Findere rule (Alg. 2).
 *   A k-mer containing a non-ACGT symbol or running past the end of its record
 *   does not exist: it is never inserted and queries false.
 *
 * Conventions
 *   - All `d_*` pointers are DEVICE pointers owned by the caller; all `h_*`
 *     pointers are HOST pointers owned by the caller.  The library owns the
 *     filter and its scratch buffers (on the device that was current at
 *     sbf_create()).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default
 *     stream).  Device-facing calls only enqueue work on `stream` and never
 *     synchronise; exception: when the internal scratch must grow,
 *     the call performs a cudaMalloc (implicitly synchronising).  Call
 *     sbf_reserve() up front to avoid that.  One call in flight per handle.
 *   - Every function returns SBF_OK (0) or a negative sbf_status; nothing
 *     throws across this boundary.  sbf_last_error() gives a message for the
 *     last failure on the calling thread.
 *   - There is no CPU fallback: without a CUDA device sbf_create() fails.
 */
#ifndef SBF_H
#define SBF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sbf sbf_t; /* opaque */

typedef enum sbf_status {
    SBF_OK = 0,
    SBF_ERR_INVALID_ARG = -1, /* NULL handle/pointer, bad sizes */
    SBF_ERR_UNSUPPORTED = -2, /* parameter combination outside what the kernels support */
    SBF_ERR_NOMEM = -3,       /* device or host allocation failed */
    SBF_ERR_CUDA = -4         /* any other CUDA runtime error (message in sbf_last_error) */
} sbf_status;

/*
 * sbf_create — allocate a zeroed filter (A8).
 *   1 <= k <= 64 (k <= 32: one 64-bit word per packed k-mer; larger k: see sbf_create_ex); 1 <= m <= k; 1 <= s <= k;
 *   1 <= H <= 32 (H <= 10 uses bit-slicing A5, H > 10 the salted multiply A6);
 *   num_bits >= 1.  numShards = next power of two >= ceil(num_bits/256), at most 2^32.
 *   Layout in device memory (A12): shard-major, four little-endian 64-bit sector words
 *   per shard, 32 bytes per shard, 32-byte aligned (one L2 sector per shard).
 *   (k,m,s,H) combinations compiled as specialised streaming kernels run those; every
 *   other legal combination runs a runtime-parameter CUDA kernel (same bits, slower).
 *   No device-wide side effects.  Only when the environment sets SBF_L2_WINDOW=1 and the filter fits the persisting L2
 *   carve-out (a7) does the call raise cudaLimitPersistingL2CacheSize (a DEVICE-wide limit) and later calls on the
 *   handle set an access-policy window for the filter on the stream they are given; measured on config 2 the window
 *   changes neither kernel times nor L2 hit rates (profiles/l2_window_r03.md), hence off by default.
 *   Returns NULL on error.
 */
sbf_t *sbf_create(int k, int m, int s, int H, uint64_t num_bits);

/*
 * sbf_create_ex — the same for any of the paper's three alphabets and for packed k-mers wider than one 64-bit
 * word ("multiword"); readings A19-A22 of DESIGN.md §3.  k * symbol_bits <= 128:
 *   SBF_ALPHABET_DNA          2 bits, A C G T either case, k <= 64 (sbf_create is this alphabet; k <= 32 runs the
 *                             specialised / runtime kernels above; 33 <= k <= 64 runs specialised streaming kernels
 *                             where an instance is compiled — e.g. (63,40,60,4), (51,31,48,4) — else the wide kernel)
 *   SBF_ALPHABET_PROTEIN      5 bits, the 26 letters either case (code = letter - 'A'), k <= 25
 *   SBF_ALPHABET_DNA_TRIPLET  6 bits, one symbol = three DNA bases (code = 16 c0 + 4 c1 + c2), k <= 21; symbols sit at
 *                             multiples of three bytes from the start of their record; k, m, s count SYMBOLS
 * All `len` / `total_bases` / offsets stay in BYTES.  Result bitmaps are indexed by the BYTE position of a k-mer's
 * first byte.  A window wider than 64 bits is folded (lo ^ rotl32(hi * 0x9E3779B97F4A7C15)) before it is hashed.
 * These run one general CUDA kernel (Alg. 1/2 as printed, one k-mer per thread): correct, not tuned — the paper
 * evaluates DNA only and calls the larger alphabets "functional".
 */
typedef enum sbf_alphabet { SBF_ALPHABET_DNA = 0, SBF_ALPHABET_PROTEIN = 1, SBF_ALPHABET_DNA_TRIPLET = 2 } sbf_alphabet;
sbf_t *sbf_create_ex(int k, int m, int s, int H, uint64_t num_bits, int alphabet);

/* sbf_destroy — free filter and scratch.  Synchronises the device.  NULL is ignored. */
void sbf_destroy(sbf_t *f);

/* Geometry of the filter actually allocated (A8): 256 * numShards bits. */
uint64_t sbf_num_bits(const sbf_t *f);
uint64_t sbf_num_shards(const sbf_t *f);
/* 1 if (k,m,s,H) runs the specialised streaming kernels, 0 if it runs the runtime-parameter kernels. */
int sbf_is_specialized(const sbf_t *f);

/* sbf_reserve — pre-size the internal scratch (2-bit packed sequence + validity mask)
 * for batches of up to max_bases symbols, so later calls never allocate. */
int sbf_reserve(sbf_t *f, uint64_t max_bases);

/* sbf_clear — zero the filter, stream-ordered. */
int sbf_clear(sbf_t *f, void *stream);

/*
 * sbf_insert_seq — insert every valid k-mer of one sequence (Alg. 1).
 *   d_seq: `len` ASCII symbols on the device.  A,C,G,T in either case are valid (A9);
 *   any other byte is invalid and k-mers covering it are skipped.  len may be 0.
 */
int sbf_insert_seq(sbf_t *f, const char *d_seq, uint64_t len, void *stream);

/*
 * sbf_insert_records — insert a dense batch of records ("dense record batch").
 *   d_bases: the records' symbols concatenated, `total_bases` bytes, no separators.
 *   d_offsets: n_rec+1 non-decreasing device uint64, d_offsets[0] = 0,
 *   d_offsets[n_rec] = total_bases; record r = d_bases[d_offsets[r] .. d_offsets[r+1]).
 *   Empty records are allowed.  No k-mer spans two records.
 *   total_bases is passed by value so the call needs no device->host read.
 */
int sbf_insert_records(sbf_t *f, const char *d_bases, const uint64_t *d_offsets, uint64_t n_rec,
                       uint64_t total_bases, void *stream);

/*
 * sbf_query_seq — query every k-mer start position of one sequence (Alg. 2).
 *   d_bitmap: ceil(len/32) device uint32 words, all written (no pre-zeroing needed):
 *   bit p (word p>>5, bit p&31) = 1 iff a valid k-mer starts at symbol p and all its
 *   H*(k-s+1) bits are set; invalid k-mers and the last k-1 positions give 0 (A11).
 *   d_hits: NULL, or one device uint64 that receives the number of set bits.
 */
int sbf_query_seq(sbf_t *f, const char *d_seq, uint64_t len, uint32_t *d_bitmap, uint64_t *d_hits,
                  void *stream);

/*
 * sbf_query_records — same for a dense record batch; bit index = position in the
 *   concatenated buffer; d_bitmap has ceil(total_bases/32) words.
 *   d_hit_counts: NULL, or n_rec device uint32: set bits of record r.
 */
int sbf_query_records(sbf_t *f, const char *d_bases, const uint64_t *d_offsets, uint64_t n_rec,
                      uint64_t total_bases, uint32_t *d_bitmap, uint32_t *d_hit_counts, void *stream);

/*
 * Host-facing forms ("host-facing calls synchronise").  The symbols (and offsets,
 * and results) live in HOST memory; the library stages them through pinned buffers in
 * chunks, overlapping the copies with the kernels on two internal streams,
 * and returns after everything has completed.  A host-facing call first waits for all work enqueued on the device
 * before it (cudaDeviceSynchronize), so it may follow device-facing calls on any stream.
 * h_bitmap / h_hit_counts as above, on the host.  For full PCIe speed every host buffer, h_offsets included, should be
 * pinned (cudaHostAlloc / cudaHostRegister): pageable symbols are staged through pinned buffers, pageable offsets and
 * results are copied at pageable speed.
 */
int sbf_insert_seq_host(sbf_t *f, const char *h_seq, uint64_t len);
int sbf_insert_records_host(sbf_t *f, const char *h_bases, const uint64_t *h_offsets, uint64_t n_rec);
int sbf_query_seq_host(sbf_t *f, const char *h_seq, uint64_t len, uint32_t *h_bitmap, uint64_t *h_hits);
int sbf_query_records_host(sbf_t *f, const char *h_bases, const uint64_t *h_offsets, uint64_t n_rec,
                           uint32_t *h_bitmap, uint32_t *h_hit_counts);

/*
 * FASTA / FASTQ text in HOST memory ("streamed FASTA/FASTQ input"; "Host FASTX staging").
 *   h_text: n_bytes of uncompressed FASTA or FASTQ text (host memory; pinned memory is copied from directly).
 *   format: 1 FASTA, 2 FASTQ, 0 = decide from the first non-blank byte ('@' -> FASTQ, anything else -> FASTA).
 *   Text rules: lines end at '\n'; '\r' is dropped; FASTA: a line starting with '>' is a header and starts a
 *   record, every other line is sequence of the current record (text before the first header is inserted by the
 *   insert call and ignored by the query call); FASTQ: four lines per record (header, sequence, '+', quality;
 *   multi-line FASTQ is not supported); a record starts at a line of index 0 mod 4 whose first byte is neither '\n'
 *   nor '\r' — a blank line, e.g. the last one of a text ending in "\n\n", counts as a line but opens no record.  Sequence bytes are taken verbatim: validity is the alphabet's (A9 / A19).
 * The raw text is copied to the device in chunks of sbf_set_host_chunk() bytes on one stream while the previous
 * chunk is normalised ON THE DEVICE (headers, quality and line ends dropped, records compacted into a dense batch +
 * offsets) and inserted / queried on another; records and k-mers may straddle chunk edges.  Synchronises.
 *   sbf_insert_fastx_host: inserts every record.  *n_records / *n_bases (nullable) receive the number of records
 *   (record starts) and of sequence bytes found.
 *   sbf_query_fastx_host: h_hit_counts[r] (nullable) = number of k-mers of record r reported present, r in file
 *   order, for r < *n_records; max_records = capacity of h_hit_counts (SBF_ERR_INVALID_ARG if the text holds more).
 */
int sbf_insert_fastx_host(sbf_t *f, const char *h_text, uint64_t n_bytes, int format, uint64_t *n_records, uint64_t *n_bases);
int sbf_query_fastx_host(sbf_t *f, const char *h_text, uint64_t n_bytes, int format, uint32_t *h_hit_counts,
                         uint64_t max_records, uint64_t *n_records, uint64_t *n_bases);

/* sbf_set_host_chunk — symbols per staged chunk of the host-facing calls ("multi-chunk workloads"):
 * a multiple of 128, larger than k + 128; default 32 Mi (the measured optimum on B200 / PCIe 5).  Chunks overlap by
 * k-1 symbols so that every k-mer lies wholly inside one chunk.  A tuning knob; tests use small chunks to put
 * record boundaries before, on and inside the overlap. */
int sbf_set_host_chunk(sbf_t *f, uint64_t symbols);

/* sbf_export_bits — copy the filter (32*numShards bytes, layout A12) to host memory.
 * nbytes must equal 32*numShards.  Synchronises the device. */
int sbf_export_bits(const sbf_t *f, void *h_dst, uint64_t nbytes);
/* sbf_import_bits — the inverse: overwrite the filter from host memory.  Synchronises. */
int sbf_import_bits(sbf_t *f, const void *h_src, uint64_t nbytes);
/* sbf_filter_device_ptr — the filter's device address (read-only use by the caller, e.g. a
 * multi-GPU OR-reduce of replicas). */
const uint64_t *sbf_filter_device_ptr(const sbf_t *f);
/* sbf_or_bits_device — filter |= d_src (32*numShards bytes on the device), stream-ordered.
 * The merge step of the replica scheme. */
int sbf_or_bits_device(sbf_t *f, const uint64_t *d_src, uint64_t nbytes, void *stream);

/* sbf_or_range_device — the same for a sub-range: filter[offset_bytes .. +nbytes) |= d_src[0 .. nbytes).
 * offset_bytes and nbytes are multiples of 32 (whole shards), d_src is 16-byte aligned.  Lets the
 * replica merge run window by window (paper_2606_24417_b200/replicas.py). */
int sbf_or_range_device(sbf_t *f, uint64_t offset_bytes, const uint64_t *d_src, uint64_t nbytes, void *stream);

/* sbf_or_peers_range_device — filter[offset_bytes .. +nbytes) |= OR over n_peers (<= 15) replicas of the SAME range,
 * each given by a device pointer to the start of its range and read in place: peer-GPU memory mapped through CUDA IPC
 * (sbf_ipc_open_filter) over NVLink, or other filters on this device.  The reduce-scatter step of the replica merge as
 * one kernel per window, without a receive buffer (paper_2606_24417_b200/replicas.py: or_allreduce_filter_peer).
 * d_peer_ranges is a HOST array of device pointers (16-byte aligned); stream-ordered. */
int sbf_or_peers_range_device(sbf_t *f, uint64_t offset_bytes, const uint64_t *const *d_peer_ranges, int n_peers, uint64_t nbytes,
                              void *stream);
/* CUDA IPC plumbing for the above: export this filter's allocation as a 64-byte handle another process (rank) of the
 * same node can open; open / close a peer's.  The mapping gives direct loads over NVLink (peer access is enabled
 * lazily).  Never executed on more than one GPU in this repository's test environment (one GPU per box). */
int sbf_ipc_export_filter(const sbf_t *f, void *handle64);
int sbf_ipc_open_filter(const void *handle64, uint64_t **d_ptr);
int sbf_ipc_close_filter(uint64_t *d_ptr);

/*
 * sbf_query_seq_static — sbf_query_seq (Alg. 2) for callers that must not allocate device memory.
 *
 * Who this is for.  A query needs working memory besides its input and output: the 2-bit packed copy of the sequence
 * and its validity mask (0.375 bytes per symbol), which the handle-based calls cudaMalloc and grow on demand.  Some
 * programs cannot let a library do that: a service whose device memory was handed out in full to its own arena or to a
 * framework's caching allocator at start-up (a cudaMalloc from a library then fails, or steals from that pool); a
 * latency-bound loop that cannot take the device-wide synchronisation a cudaMalloc / cudaFree implies; a plug-in that
 * runs under a fixed per-process memory budget (MPS / MIG partitions) and may only use what its host hands it.  Such a
 * caller keeps the filter in memory of its own and calls this one function: no handle, no cudaMalloc, cudaFree,
 * cudaMallocAsync or any other allocating routine, on any call.
 *
 * Working memory.  The packed copy and the mask live in ONE array of device memory compiled into the library
 * (6 MiB + 512 bytes, file scope in sbf_api.cu).  Every GPU whose context loads libsbf_b200.so holds that array from module
 * load until the process exits, whether or not this function is ever called.  Its size fixes the limit:
 *   len <= SBF_STATIC_MAX_SYMBOLS (2^24 = 16 Mi symbols per call); a longer sequence is rejected with
 *   SBF_ERR_INVALID_ARG and a message that names the limit — split it into pieces that overlap by k-1 symbols.
 *
 * Arguments (all device pointers are the caller's, on the CURRENT device):
 *   k, m, s, H      as sbf_create; DNA alphabet only.  k <= 32, or 33 <= k <= 64 where a streaming instance is compiled;
 *                   anything else is SBF_ERR_UNSUPPORTED (the other alphabets' kernel needs no working memory at all,
 *                   so sbf_query_seq on a handle already allocates nothing for them).
 *   d_filter        the filter in layout A12: num_shards x 32 bytes, 32-byte aligned, read only.  num_shards is a power
 *                   of two, at most 2^32, and must be the shard count the bits were inserted with.  Either memory the
 *                   caller filled itself (e.g. from sbf_export_bits of another process) or sbf_filter_device_ptr() /
 *                   sbf_num_shards() of a handle created while allocating was still allowed.
 *   d_seq, len      the ASCII symbols, as sbf_query_seq.  len may be 0 (nothing is enqueued).
 *   d_bitmap        ceil(len/32) uint32 words, all written; bit p as in sbf_query_seq.
 *   stream          the work is enqueued on it and the call returns without synchronising.
 *
 * Set-up.  The FIRST call on each device looks up the device address of the array (once per device, with that device
 * current; the result is cached) before it enqueues anything.  Make that first call outside any stream capture, e.g.
 * with len = 0 at start-up; later calls on the same device only launch kernels.
 *
 * Sharing.  All calls in the process — every thread, every stream, every filter — use the same array, and it keeps
 * whatever the previous call left in it.  That is harmless in sequence: the packing step rewrites every word the query
 * step reads before it reads it, so nothing has to start at zero and nothing is cleared.  It is NOT harmless in
 * parallel: two calls whose kernels may overlap on one GPU (different streams, or different host threads) race on the
 * array and both results are undefined.  Order such calls on one stream or with events.  Calls on different GPUs do not
 * interact (each GPU has its own copy).  The handle-based calls never touch this array.
 *
 * Result: bit-identical to sbf_query_seq on a handle with the same (k,m,s,H) and filter contents.  The L2 persistence
 * window of a7 is not applied (stream attributes are left alone).
 */
#define SBF_STATIC_MAX_SYMBOLS (1ull << 24)
int sbf_query_seq_static(int k, int m, int s, int H, const uint64_t *d_filter, uint64_t num_shards, const char *d_seq,
                         uint64_t len, uint32_t *d_bitmap, void *stream);

/* Message for the last error on the calling thread ("" if none). */
const char *sbf_last_error(void);

/* Counts kernels launched by this library in this process (all handles); bench.py reports it. */
uint64_t sbf_kernel_launches(void);

/* sbf_set_timing — on != 0: every later device-facing insert/query call on this handle records CUDA
 * events on the caller's stream around each kernel it enqueues (a few microseconds per call).
 * sbf_get_timing — device time of the kernels of the LAST such call, in milliseconds:
 *   ms3[0] = pack (+ record-end marking), ms3[1] = the fused insert or query kernel,
 *   ms3[2] = the hit-count kernel (0 when none ran).  Waits for that call's last event.
 * bench.py uses these for the per-kernel roofline figures. */
int sbf_set_timing(sbf_t *f, int on);
int sbf_get_timing(sbf_t *f, float *ms3);

/* The measured-ceiling micro-benchmarks (sbf_ceiling_...) and the pack test hook are not part of this boundary: they are
 * declared in include/sbf_bench.h and live in a library of their own (libsbf_bench_b200.so) that only bench.py and the
 * tests load. */

#ifdef __cplusplus
}
#endif
#endif /* SBF_H */

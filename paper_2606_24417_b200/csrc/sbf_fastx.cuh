// sbf_fastx.cuh — FASTA / FASTQ normalisation on the device ("Host FASTX staging").
//
// The paper normalises FASTX text on the host and stages the result; here the raw text crosses PCIe once, chunk by
// chunk, and is normalised where it lands: header / quality lines and line ends are dropped, the sequence bytes are
// compacted into the dense record batch + offsets that sbf_insert_records / sbf_query_records take ("dense
// record batch"), with the lexer state carried from chunk to chunk in device memory.
//
// Text rules (the oracle side restates them in oracle/fastx.py):
//   lines end at '\n'; '\r' is never a sequence byte; every other byte of a sequence line is copied verbatim
//   FASTA  a line whose first byte is '>' is a header and starts a record; all other lines are sequence lines of the
//          current record (bytes before the first header belong to "record 0" of the chunk, see below)
//   FASTQ  four lines per record: header, sequence, '+', quality (line index mod 4; multi-line FASTQ is not supported);
//          a record starts at the first byte of a line with index = 0 mod 4, unless that byte is '\n' or '\r' (a blank
//          line, e.g. the second '\n' of a text ending in "\n\n", still counts as a line but opens no record)
// One chunk of text yields: dense bytes [carry | sequence bytes of the chunk], offsets[0] = 0, one offset per record
// start, offsets[n_rec] = n_bases, with n_rec = 1 + record starts: local record 0 is whatever precedes the first
// record start of the chunk — the continuation of the previous chunk's last record, led by its last k-1 bytes (the
// carry), so that k-mers straddling a chunk edge are seen exactly once.
//
// Three launches per chunk, all plain integer scans over 16 KiB tiles:
//   fastx_tile_kernel  per tile, a summary that composes associatively (see Seg)
//   fastx_scan_kernel  one thread: exclusive prefix over the tile summaries, totals, next chunk's lexer state
//   fastx_emit_kernel  per tile: the same summaries per thread, scanned inside the tile, then every thread writes
//                      the sequence bytes and record starts of its 64 bytes at their final positions
#pragma once

#include <cstdint>
#include <cuda_runtime.h>

namespace sbfk {

constexpr int kFxThreads = 256;
constexpr int kFxPerThread = 64;
constexpr int kFxTile = kFxThreads * kFxPerThread; // 16 KiB of text per CTA

enum { kFxFasta = 1, kFxFastq = 2 };

struct FastxState {          // device-resident, carried from one chunk to the next
    uint32_t at_line_start;  // the chunk's first byte begins a line
    uint32_t in_header;      // FASTA: the chunk starts inside a header line
    uint32_t line_mod4;      // FASTQ: index of the line the chunk starts in, mod 4
    uint32_t carry_len;      // bytes already at the front of the dense buffer (tail of the previous chunk's last record)
    uint64_t n_bases;        // out: bytes in the dense buffer, carry included
    uint64_t n_starts;       // out: record starts in this chunk (offsets has n_starts + 2 entries)
};

// Summary of a stretch of text; compose(A, B) is the summary of A followed by B (associative, not commutative).
//   FASTA: has_ls/last_hdr = the stretch contains a line start / its last line start is a header; pre = non-EOL bytes
//          before the first line start (sequence iff the stretch is entered outside a header); post = sequence bytes
//          after it (decided locally); starts = header line starts.
//   FASTQ: nl = newlines; seq[r] = non-EOL bytes on lines whose local index is r mod 4; ls[r] = starts of non-blank lines with
//          local index r mod 4 (local index = newlines before the byte).
struct Seg {
    uint32_t has_ls, last_hdr, pre, post, starts; // FASTA
    uint32_t nl, seq[4], ls[4];                   // FASTQ
};

template <int FMT>
__device__ __forceinline__ Seg seg_identity()
{
    Seg s;
    s.has_ls = s.last_hdr = s.pre = s.post = s.starts = 0;
    s.nl = 0;
#pragma unroll
    for (int r = 0; r < 4; ++r) { s.seq[r] = 0; s.ls[r] = 0; }
    return s;
}

template <int FMT>
__device__ __forceinline__ Seg seg_compose(const Seg &a, const Seg &b)
{
    Seg c = seg_identity<FMT>();
    if (FMT == kFxFasta) {
        c.has_ls = a.has_ls | b.has_ls;
        c.last_hdr = b.has_ls ? b.last_hdr : a.last_hdr;
        c.pre = a.has_ls ? a.pre : a.pre + b.pre;
        c.post = a.post + b.post + ((a.has_ls && !a.last_hdr) ? b.pre : 0);
        c.starts = a.starts + b.starts;
    } else {
        c.nl = a.nl + b.nl;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            c.seq[r] = a.seq[r] + b.seq[(r - (int)a.nl) & 3];
            c.ls[r] = a.ls[r] + b.ls[(r - (int)a.nl) & 3];
        }
    }
    return c;
}

// what a stretch contributes when it is entered in lexer state st: sequence bytes, record starts
template <int FMT>
__device__ __forceinline__ void seg_apply(const Seg &s, const FastxState &st, uint32_t &n_seq, uint32_t &n_starts)
{
    if (FMT == kFxFasta) {
        n_seq = (st.in_header ? 0 : s.pre) + s.post;
        n_starts = s.starts;
    } else {
        n_seq = s.seq[(1 - (int)st.line_mod4) & 3];
        n_starts = s.ls[(0 - (int)st.line_mod4) & 3];
    }
}
// lexer state after the stretch
template <int FMT>
__device__ __forceinline__ void seg_advance(const Seg &s, FastxState &st)
{
    if (FMT == kFxFasta) {
        if (s.has_ls) st.in_header = s.last_hdr;
    } else {
        st.line_mod4 = (st.line_mod4 + s.nl) & 3;
    }
}

__device__ __forceinline__ bool fx_is_eol(uint8_t c) { return c == '\n' || c == '\r'; }

// summary of text[i0, i1) (i1 <= n); prev = the byte before i0 ('\n' if the stretch starts a line)
template <int FMT>
__device__ __forceinline__ Seg seg_of(const uint8_t *__restrict__ text, uint64_t i0, uint64_t i1, uint8_t prev)
{
    Seg s = seg_identity<FMT>();
    bool hdr_line = false; // FASTA: the line we are in started inside this stretch and is a header
    for (uint64_t i = i0; i < i1; ++i) {
        const uint8_t c = text[i];
        const bool ls = prev == '\n';
        if (FMT == kFxFasta) {
            if (ls) {
                hdr_line = c == '>';
                s.has_ls = 1;
                s.last_hdr = hdr_line;
                s.starts += hdr_line;
            }
            if (!fx_is_eol(c)) {
                if (!s.has_ls) ++s.pre;
                else if (!hdr_line) ++s.post;
            }
        } else {
            if (ls && !fx_is_eol(c)) ++s.ls[s.nl & 3]; // a blank line opens no record
            if (!fx_is_eol(c)) ++s.seq[s.nl & 3];
            if (c == '\n') ++s.nl;
        }
        prev = c;
    }
    return s;
}

#ifdef SBF_DEFINE_AUX_KERNELS

// ordered reduction / exclusive scan of one Seg per thread inside a CTA of kFxThreads: lane 0 of each warp composes its
// 32 entries, thread 0 the 8 warp results.  sm holds kFxThreads + 8 entries.  On return mine = the composition of the
// entries of all threads before this one; the return value (valid in every thread) is the whole tile's summary.
template <int FMT>
__device__ Seg block_exclusive_scan(Seg &mine, Seg *sm)
{
    const int t = threadIdx.x, w = t >> 5;
    sm[t] = mine;
    __syncthreads();
    if ((t & 31) == 0) {
        Seg acc = seg_identity<FMT>();
        for (int j = 0; j < 32; ++j) {
            const Seg cur = sm[t + j];
            sm[t + j] = acc; // exclusive prefix inside the warp
            acc = seg_compose<FMT>(acc, cur);
        }
        sm[kFxThreads + w] = acc;
    }
    __syncthreads();
    if (t == 0) {
        Seg acc = seg_identity<FMT>();
        for (int j = 0; j < kFxThreads / 32; ++j) {
            const Seg cur = sm[kFxThreads + j];
            sm[kFxThreads + j] = acc;
            acc = seg_compose<FMT>(acc, cur);
        }
        sm[kFxThreads + 8] = acc;
    }
    __syncthreads();
    mine = seg_compose<FMT>(sm[kFxThreads + w], sm[t]);
    return sm[kFxThreads + 8];
}

template <int FMT>
__global__ void __launch_bounds__(kFxThreads) fastx_tile_kernel(const uint8_t *__restrict__ text, uint64_t n, const FastxState *st,
                                                                Seg *tile_sum)
{
    __shared__ Seg sm[kFxThreads + 9];
    const uint64_t i0 = (uint64_t)blockIdx.x * kFxTile + (uint64_t)threadIdx.x * kFxPerThread;
    const uint64_t i1 = i0 + kFxPerThread < n ? i0 + kFxPerThread : n;
    Seg mine = seg_identity<FMT>();
    if (i0 < n) mine = seg_of<FMT>(text, i0, i1, i0 == 0 ? (st->at_line_start ? '\n' : 'x') : text[i0 - 1]);
    const Seg total = block_exclusive_scan<FMT>(mine, sm);
    if (threadIdx.x == 0) tile_sum[blockIdx.x] = total;
}

// exclusive prefix over the tiles (in place), totals and the lexer state of the next chunk -> *st_next; offsets[0] and
// offsets[n_starts + 1] of this chunk.
template <int FMT>
__global__ void fastx_scan_kernel(Seg *tile_sum, uint32_t n_tiles, const uint8_t *__restrict__ text, uint64_t n, FastxState *st,
                                  FastxState *st_next, uint64_t *offsets)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    Seg acc = seg_identity<FMT>();
    for (uint32_t t = 0; t < n_tiles; ++t) {
        const Seg cur = tile_sum[t];
        tile_sum[t] = acc;
        acc = seg_compose<FMT>(acc, cur);
    }
    uint32_t n_seq, n_starts;
    seg_apply<FMT>(acc, *st, n_seq, n_starts);
    st->n_bases = (uint64_t)st->carry_len + n_seq;
    st->n_starts = n_starts;
    offsets[0] = 0;
    offsets[(uint64_t)n_starts + 1] = st->n_bases;
    FastxState nx = *st;
    seg_advance<FMT>(acc, nx);
    nx.at_line_start = n == 0 ? st->at_line_start : (text[n - 1] == '\n');
    nx.carry_len = 0; // set by fastx_carry_kernel
    nx.n_bases = 0; nx.n_starts = 0;
    *st_next = nx;
}

template <int FMT>
__global__ void __launch_bounds__(kFxThreads) fastx_emit_kernel(const uint8_t *__restrict__ text, uint64_t n, const FastxState *st,
                                                                const Seg *tile_pre, uint8_t *__restrict__ dense,
                                                                uint64_t *__restrict__ offsets)
{
    __shared__ Seg sm[kFxThreads + 9];
    const uint64_t i0 = (uint64_t)blockIdx.x * kFxTile + (uint64_t)threadIdx.x * kFxPerThread;
    const uint64_t i1 = i0 + kFxPerThread < n ? i0 + kFxPerThread : n;
    const uint8_t prev0 = i0 == 0 ? (st->at_line_start ? '\n' : 'x') : (i0 < n ? text[i0 - 1] : 'x');
    Seg mine = seg_identity<FMT>();
    if (i0 < n) mine = seg_of<FMT>(text, i0, i1, prev0);
    (void)block_exclusive_scan<FMT>(mine, sm);
    if (i0 >= n) return;
    // everything before this thread's bytes: the tiles before this one, then the threads before this one
    const Seg before = seg_compose<FMT>(tile_pre[blockIdx.x], mine);
    FastxState cur = *st;
    uint32_t n_seq, n_starts;
    seg_apply<FMT>(before, cur, n_seq, n_starts);
    seg_advance<FMT>(before, cur);
    uint64_t pos = (uint64_t)cur.carry_len + n_seq; // dense position of this thread's first sequence byte
    uint64_t rec = n_starts;                        // record starts before it
    bool in_hdr = cur.in_header != 0;
    uint32_t line = cur.line_mod4;
    uint8_t prev = prev0;
    for (uint64_t i = i0; i < i1; ++i) {
        const uint8_t c = text[i];
        const bool ls = prev == '\n';
        bool is_seq;
        if (FMT == kFxFasta) {
            if (ls) {
                in_hdr = c == '>';
                if (in_hdr) offsets[1 + rec++] = pos;
            }
            is_seq = !in_hdr && !fx_is_eol(c);
        } else {
            if (ls && line == 0 && !fx_is_eol(c)) offsets[1 + rec++] = pos;
            is_seq = line == 1 && !fx_is_eol(c);
            if (c == '\n') line = (line + 1) & 3;
        }
        if (is_seq) dense[pos++] = c;
        prev = c;
    }
}

// the last min(k_bytes - 1, length) bytes of the chunk's last record -> front of the next chunk's dense buffer
__global__ void fastx_carry_kernel(const uint8_t *__restrict__ dense, const uint64_t *__restrict__ offsets, const FastxState *st,
                                   uint32_t keep, uint8_t *__restrict__ next_dense, FastxState *st_next)
{
    const uint64_t last_start = offsets[st->n_starts];
    const uint64_t len = st->n_bases - last_start;
    const uint32_t cl = len < (uint64_t)keep ? (uint32_t)len : keep;
    for (uint32_t j = threadIdx.x; j < cl; j += blockDim.x) next_dense[j] = dense[st->n_bases - cl + j];
    if (threadIdx.x == 0) st_next->carry_len = cl;
}

// per-record hit counts of one chunk added into the batch's counts: local record i is global record base - 1 + i (local
// record 0 continues the previous chunk's last record; with base == 0 it is the text before the first record: dropped)
__global__ void __launch_bounds__(256) fastx_add_counts_kernel(const uint32_t *__restrict__ local, uint64_t n_local, uint64_t base,
                                                               uint32_t *__restrict__ global, uint64_t max_records)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_local; i += (uint64_t)gridDim.x * blockDim.x) {
        if (i == 0 && base == 0) continue;
        const uint64_t g = base - 1 + i;
        if (g < max_records) global[g] += local[i]; // one writer per slot: records of one chunk are distinct
    }
}

#endif // SBF_DEFINE_AUX_KERNELS

} // namespace sbfk

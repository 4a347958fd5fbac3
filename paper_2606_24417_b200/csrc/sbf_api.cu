// sbf_api.cu — the C ABI of include/sbf.h: handle, scratch, kernel dispatch, host-facing staging.
// Every step of the path (pack, minimizer, shard, s-mer hashing, merge, result bitmap, hit counts)
// runs in the kernels of sbf_device.cuh; this file only sizes buffers and enqueues launches.
#include "../../include/sbf.h"

#include <algorithm>
#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#define SBF_DEFINE_AUX_KERNELS
#include "sbf_dispatch.h"
#include "sbf_fastx.cuh"

using namespace sbfk;

namespace {

constexpr uint64_t kHostChunkDefault = 32ull << 20; // host-facing path: symbols per staged chunk, multiple of 128 (measured best of 8..128 Mi)

// insert: from this filter size on a run is flushed with one 32-byte TMA reduction instead of four RED.OR.B64
// (measured per 100 Mbp on B200: 2^31 bits 0.48 vs 0.50 ms, 2^32 bits 0.49 vs 0.57 ms, 2^35 bits 0.58 vs 0.70 ms; 2^30 bits 0.48 vs 0.38 ms)
#ifndef SBF_TMA_MIN_BYTES
#define SBF_TMA_MIN_BYTES (256ull << 20)
#endif
constexpr uint64_t kTmaFlushMinBytes = SBF_TMA_MIN_BYTES;

thread_local std::string g_err;
std::atomic<uint64_t> g_launches{0};

int fail(int code, const char *what)
{
    g_err = what;
    return code;
}
int fail_cuda(cudaError_t e, const char *where)
{
    g_err = std::string(where) + ": " + cudaGetErrorString(e);
    return e == cudaErrorMemoryAllocation ? SBF_ERR_NOMEM : SBF_ERR_CUDA;
}
#define CK(call)                                                  \
    do {                                                          \
        cudaError_t e__ = (call);                                 \
        if (e__ != cudaSuccess) return fail_cuda(e__, #call);     \
    } while (0)

struct TableList { // filled by the static TableRegistration objects of the sbf_inst_*.cu objects at load time
    const KernelEntry *entries[64];
    int counts[64];
    int n;
};
TableList &tables()
{
    static TableList t = {};
    return t;
}

const KernelEntry *find_entry(int k, int m, int s, int H)
{
    const TableList &t = tables();
    for (int i = 0; i < t.n; ++i)
        for (int j = 0; j < t.counts[i]; ++j) {
            const KernelEntry &e = t.entries[i][j];
            if (e.k == k && e.m == m && e.s == s && e.H == H) return &e;
        }
    return nullptr;
}

struct HostRun { // persistent state of the host-facing path (two slots: copy c+1 while computing c)
    cudaStream_t copy = nullptr, comp = nullptr;
    cudaEvent_t copied[2] = {nullptr, nullptr}, computed[2] = {nullptr, nullptr}, offs_ready = nullptr;
    char *pin[2] = {nullptr, nullptr};     // pinned staging for symbols (pageable caller memory only)
    char *d_bases[2] = {nullptr, nullptr};
    uint64_t *d_off[2] = {nullptr, nullptr};
    uint64_t cap_pin = 0, cap_bases = 0, cap_off = 0;
    uint32_t *d_bitmap = nullptr;  uint64_t cap_bitmap = 0;
    uint64_t *d_off_full = nullptr; uint32_t *d_counts = nullptr; uint64_t cap_rec = 0;
    unsigned long long *d_hits = nullptr;
    ~HostRun()
    {
        for (int i = 0; i < 2; ++i) {
            if (copied[i]) cudaEventDestroy(copied[i]);
            if (computed[i]) cudaEventDestroy(computed[i]);
            if (pin[i]) cudaFreeHost(pin[i]);
            if (d_bases[i]) cudaFree(d_bases[i]);
            if (d_off[i]) cudaFree(d_off[i]);
        }
        if (offs_ready) cudaEventDestroy(offs_ready);
        if (d_bitmap) cudaFree(d_bitmap);
        if (d_off_full) cudaFree(d_off_full);
        if (d_counts) cudaFree(d_counts);
        if (d_hits) cudaFree(d_hits);
        if (copy) cudaStreamDestroy(copy);
        if (comp) cudaStreamDestroy(comp);
        cudaGetLastError();
    }
};

struct FastxRun { // persistent state of the FASTX host path (two slots: copy chunk c+1 while chunk c is normalised and walked)
    cudaStream_t copy = nullptr, comp = nullptr;
    cudaEvent_t copied[2] = {nullptr, nullptr}, computed[2] = {nullptr, nullptr}, normalised = nullptr;
    char *pin[2] = {nullptr, nullptr};
    uint8_t *d_text[2] = {nullptr, nullptr}, *d_dense[2] = {nullptr, nullptr};
    uint64_t *d_off[2] = {nullptr, nullptr};
    uint64_t cap_text = 0; // bytes of text per slot the buffers above are sized for
    Seg *d_tiles = nullptr;
    FastxState *d_state = nullptr, *h_state = nullptr; // 2 device states (alternating), one pinned host copy
    uint32_t *d_bitmap = nullptr, *d_counts_local = nullptr, *d_counts = nullptr;
    uint64_t cap_counts = 0;
    ~FastxRun()
    {
        for (int i = 0; i < 2; ++i) {
            if (copied[i]) cudaEventDestroy(copied[i]);
            if (computed[i]) cudaEventDestroy(computed[i]);
            if (pin[i]) cudaFreeHost(pin[i]);
            if (d_text[i]) cudaFree(d_text[i]);
            if (d_dense[i]) cudaFree(d_dense[i]);
            if (d_off[i]) cudaFree(d_off[i]);
        }
        if (normalised) cudaEventDestroy(normalised);
        if (d_tiles) cudaFree(d_tiles);
        if (d_state) cudaFree(d_state);
        if (h_state) cudaFreeHost(h_state);
        if (d_bitmap) cudaFree(d_bitmap);
        if (d_counts_local) cudaFree(d_counts_local);
        if (d_counts) cudaFree(d_counts);
        if (copy) cudaStreamDestroy(copy);
        if (comp) cudaStreamDestroy(comp);
        cudaGetLastError();
    }
};

} // namespace

namespace sbfk {
void register_table(const KernelEntry *entries, int n)
{
    TableList &t = tables();
    if (t.n < 64) {
        t.entries[t.n] = entries;
        t.counts[t.n] = n;
        ++t.n;
    }
}
} // namespace sbfk

struct sbf {
    int k, m, s, H, P;
    int device;
    uint64_t num_shards;
    uint64_t *filter;        // 4 * num_shards words
    const KernelEntry *entry; // nullptr -> runtime-parameter kernels
    bool tma_flush;           // insert flushes runs with TMA reductions (filter much larger than L2)
    // wide path (A19-A22): other alphabets, packed k-mers wider than 64 bits -> wide_tile_kernel, no pack pass
    int alphabet, sym_bits, sym_bytes;
    bool wide;
    int phase0;               // host-facing chunks only: see WideParams::phase0
    // scratch of the last batch
    uint32_t *packed;
    uint16_t *gmask;
    uint64_t cap_words;       // allocated words in packed / gmask
    uint64_t last_words;      // words written by the last pack
    uint32_t *d_flag;         // [0] record-mode fallback flag of the last query, [1] its long-record group counter (cleared by pack_kernel, raised by stream_rec_kernel)
    uint2 *d_long;            // kLongCap (record, group) entries: the long records of the last record-mode query
    // L2 persistence window (a7)
    bool l2_window;
    cudaStream_t l2_stream_set;
    bool l2_stream_valid;
    // host-facing staging (created on first use)
    HostRun *host;
    FastxRun *fastx;          // FASTX host path (created on first use)
    uint64_t host_chunk;      // symbols per staged chunk (sbf_set_host_chunk; default kHostChunkDefault)
    // optional per-kernel timing (sbf_set_timing): events on the caller's stream around each kernel
    bool timing;
    cudaEvent_t tev[4]; // before pack, after pack, after main kernel, after count kernel
    bool tev_count;     // the last call enqueued a count kernel
    bool tev_valid;     // a timed call has completed its enqueue
};

namespace {

uint64_t words_for(uint64_t n_bases) { return (n_bases + 15) / 16 + kPadWords; }

int ensure_scratch(sbf *f, uint64_t n_bases)
{
    uint64_t need = words_for(n_bases);
    if (need <= f->cap_words) return SBF_OK;
    if (f->packed) cudaFree(f->packed);
    if (f->gmask) cudaFree(f->gmask);
    f->packed = nullptr; f->gmask = nullptr; f->cap_words = 0;
    uint64_t cap = need + need / 8;
    CK(cudaMalloc(&f->packed, cap * sizeof(uint32_t)));
    CK(cudaMalloc(&f->gmask, cap * sizeof(uint16_t) + 8));
    f->cap_words = cap;
    return SBF_OK;
}

// a7: keep a filter that fits in L2 resident there (accessPolicyWindow on the caller's stream)
void apply_l2_window(sbf *f, cudaStream_t st)
{
    if (!f->l2_window) return;
    if (f->l2_stream_valid && f->l2_stream_set == st) return;
    cudaStreamAttrValue v;
    memset(&v, 0, sizeof(v));
    v.accessPolicyWindow.base_ptr = f->filter;
    v.accessPolicyWindow.num_bytes = f->num_shards * 32;
    v.accessPolicyWindow.hitRatio = 1.0f;
    v.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
    v.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
    if (cudaStreamSetAttribute(st, cudaStreamAttributeAccessPolicyWindow, &v) != cudaSuccess) {
        cudaGetLastError();
        f->l2_window = false;
        return;
    }
    f->l2_stream_set = st;
    f->l2_stream_valid = true;
}

// a1: pack + validity mask of one batch into the scratch.  Chunk mode over records (rec_bitmap == nullptr) also marks the
// record ends; record mode (rec_bitmap = the result bitmap) bounds each record by its length instead, and has the
// pack kernel zero the bitmap and the fallback flag in passing.
int run_pack(sbf *f, const char *d_bases, const uint64_t *d_offsets, uint64_t n_rec, uint64_t total, cudaStream_t st,
             uint32_t *rec_bitmap = nullptr)
{
    int rc = ensure_scratch(f, total);
    if (rc) return rc;
    uint64_t nw = words_for(total);
    f->last_words = nw;
    unsigned blocks = (unsigned)(((nw + 1) / 2 + 255) / 256);
    int aligned = ((reinterpret_cast<uintptr_t>(d_bases) & 15) == 0) ? 1 : 0;
    pack_kernel<<<blocks, 256, 0, st>>>(reinterpret_cast<const uint8_t *>(d_bases), total, f->packed, f->gmask, nw, f->k,
                                        aligned, rec_bitmap, (total + 31) / 32, rec_bitmap ? f->d_flag : nullptr);
    CK(cudaGetLastError());
    g_launches++;
    if (!rec_bitmap && d_offsets && n_rec > 1 && f->k >= 2 && total > 0) {
        unsigned b2 = (unsigned)((n_rec + 255) / 256 < 4736 ? (n_rec + 255) / 256 : 4736);
        mark_ends_kernel<<<b2, 256, 0, st>>>(d_offsets, n_rec, total, reinterpret_cast<uint32_t *>(f->gmask), f->k, nullptr);
        CK(cudaGetLastError());
        g_launches++;
    }
    return SBF_OK;
}

StreamParams make_params(sbf *f, uint64_t total, uint32_t *bitmap)
{
    StreamParams p;
    p.packed = f->packed;
    p.vmask = f->gmask;
    p.n_pos = total;
    p.filter = f->filter;
    p.shard_shift = 32 - f->P;
    p.bitmap = bitmap;
    p.n_bitmap_words = (total + 31) / 32;
    // short chunks for small batches, so that the grid still fills 148 SMs x 6 CTAs a few times over
    p.chunk_blocks = total >= (64ull << 20) ? 8 : total >= (16ull << 20) ? 4 : 2;
    p.offsets = nullptr; p.n_rec = 0; p.counts = nullptr; p.fallback = nullptr; p.rec_limit = 0;
    p.long_groups = nullptr; p.long_cap = 0;
    return p;
}

template <bool INSERT>
int run_main(sbf *f, uint64_t total, uint32_t *bitmap, cudaStream_t st)
{
    if (total == 0) return SBF_OK;
    StreamParams p = make_params(f, total, bitmap);
    if (f->entry) {
        CK((INSERT ? (f->tma_flush ? f->entry->insert_tma : f->entry->insert) : f->entry->query)(p, st));
    } else {
        if (f->k > 32) return fail(SBF_ERR_UNSUPPORTED, "internal: naive_kernel packs a k-mer into one 64-bit word (k <= 32)");
        NaiveParams np;
        np.sp = p; np.k = f->k; np.m = f->m; np.s = f->s; np.H = f->H;
        uint64_t n32 = (total + 31) / 32 * 32;
        unsigned blocks = (unsigned)((n32 + 255) / 256);
        naive_kernel<INSERT><<<blocks, 256, 0, st>>>(np);
        CK(cudaGetLastError());
    }
    g_launches++;
    return SBF_OK;
}

int mark(sbf *f, int i, cudaStream_t st)
{
    if (!f->timing) return SBF_OK;
    if (i == 0) { f->tev_count = false; f->tev_valid = false; }
    if (i == 2) f->tev_valid = true;
    if (i == 3) f->tev_count = true;
    CK(cudaEventRecord(f->tev[i], st));
    return SBF_OK;
}

// wide path: one kernel straight from the ASCII bytes (marks 0 -> 1 -> 2 keep the timing ABI's shape: "pack" = 0)
template <bool INSERT>
int run_wide(sbf *f, const char *d_bases, const uint64_t *d_offsets, uint64_t n_rec, uint64_t total, uint32_t *bitmap,
             cudaStream_t st)
{
    int rc = mark(f, 0, st);
    if (rc) return rc;
    rc = mark(f, 1, st);
    if (rc) return rc;
    WideParams p;
    p.bases = reinterpret_cast<const uint8_t *>(d_bases); p.total = total;
    p.offsets = (d_offsets && n_rec > 0) ? d_offsets : nullptr; p.n_rec = n_rec;
    p.filter = f->filter; p.shard_shift = 32 - f->P; p.bitmap = bitmap; p.n_bitmap_words = (total + 31) / 32;
    p.k = f->k; p.m = f->m; p.s = f->s; p.H = f->H; p.alphabet = f->alphabet; p.sym_bits = f->sym_bits; p.sym_bytes = f->sym_bytes;
    p.phase0 = f->phase0;
    const unsigned tiles = (unsigned)((total + kWtTile - 1) / kWtTile);
    if (p.sym_bytes == 3) wide_tile_kernel<INSERT, 3><<<tiles, kWtTPB, 0, st>>>(p);
    else wide_tile_kernel<INSERT, 1><<<tiles, kWtTPB, 0, st>>>(p);
    CK(cudaGetLastError());
    g_launches++;
    return mark(f, 2, st);
}

int run_insert(sbf *f, const char *d_bases, const uint64_t *d_offsets, uint64_t n_rec, uint64_t total, cudaStream_t st)
{
    if (total == 0) return SBF_OK;
    apply_l2_window(f, st);
    if (f->wide) return run_wide<true>(f, d_bases, d_offsets, n_rec, total, nullptr, st);
    int rc = mark(f, 0, st);
    if (rc) return rc;
    rc = run_pack(f, d_bases, d_offsets, n_rec, total, st);
    if (rc) return rc;
    rc = mark(f, 1, st);
    if (rc) return rc;
    rc = run_main<true>(f, total, nullptr, st);
    if (rc) return rc;
    return mark(f, 2, st);
}

int run_count_records(const uint32_t *d_bitmap, const uint64_t *d_offsets, uint64_t n_rec, uint64_t total, uint32_t *d_counts,
                      cudaStream_t st, const uint32_t *only_if = nullptr)
{
    if (n_rec == 0) return SBF_OK;
    if (total / n_rec < 2048) {
        unsigned blocks = (unsigned)((n_rec + 255) / 256);
        if (only_if != nullptr && blocks > 148 * 8) blocks = 148 * 8; // fallback behind record mode: strides
        count_records_thread_kernel<<<blocks, 256, 0, st>>>(d_bitmap, d_offsets, n_rec, d_counts, only_if);
    } else {
        unsigned blocks = (unsigned)(n_rec < 4096 ? n_rec : 4096);
        count_records_block_kernel<<<blocks, 256, 0, st>>>(d_bitmap, d_offsets, n_rec, d_counts);
    }
    CK(cudaGetLastError());
    g_launches++;
    return SBF_OK;
}

// Record mode (one thread per record, stream_rec_kernel) is tried for batches of short records: the host knows only
// the MEAN length.  A thread that meets a record above kRecMaxLimit lists it instead of walking it, and
// stream_long_kernel, queued right behind, walks only the listed records chunk by chunk (it exits at once when the list
// is empty).  Only when the list overflows (more than kLongCap groups) is the device flag raised, and the chunk-mode
// launches queued behind (record-end marking, chunk kernel, count kernel) then redo the whole batch; while the flag is
// clear they exit at once.  No host synchronisation either way.
constexpr uint64_t kRecMeanLimit = 400; // symbols
constexpr uint32_t kRecMaxLimit = 1024; // symbols
// list of the long records' chunk groups (128 chunks of 128 positions each): 65536 groups = 1 Gi positions of long records
constexpr uint32_t kLongCap = 65536;

int run_query(sbf *f, const char *d_bases, const uint64_t *d_offsets, uint64_t n_rec, uint64_t total, uint32_t *d_bitmap,
              uint32_t *d_counts, cudaStream_t st)
{
    if (total == 0) return SBF_OK;
    apply_l2_window(f, st);
    if (f->wide) {
        int rcw = run_wide<false>(f, d_bases, d_offsets, n_rec, total, d_bitmap, st);
        if (rcw) return rcw;
        if (d_counts && d_offsets && n_rec) {
            rcw = run_count_records(d_bitmap, d_offsets, n_rec, total, d_counts, st);
            if (rcw) return rcw;
            rcw = mark(f, 3, st);
        }
        return rcw;
    }
    const bool try_rec = f->entry && f->entry->query_rec && d_offsets && n_rec > 0 && total / n_rec <= kRecMeanLimit;
    int rc = mark(f, 0, st);
    if (rc) return rc;
    rc = run_pack(f, d_bases, d_offsets, n_rec, total, st, try_rec ? d_bitmap : nullptr);
    if (rc) return rc;
    rc = mark(f, 1, st);
    if (rc) return rc;
    if (try_rec) {
        StreamParams p = make_params(f, total, d_bitmap);
        p.offsets = d_offsets; p.n_rec = n_rec; p.counts = d_counts; p.fallback = f->d_flag; p.rec_limit = kRecMaxLimit;
        if (n_rec <= 0xFFFFFFFFull) { p.long_groups = f->d_long; p.long_cap = kLongCap; } // the list holds 32-bit record indices
        CK(f->entry->query_rec(p, st));
        g_launches++;
        if (p.long_groups) {
            CK(f->entry->query_long(p, st));
            g_launches++;
        }
        rc = mark(f, 2, st);
        if (rc) return rc;
        // the fallback behind record mode: all three exit at once unless a record was longer than kRecMaxLimit
        if (f->k >= 2 && n_rec > 1) {
            unsigned b2 = (unsigned)((n_rec + 255) / 256 < 1184 ? (n_rec + 255) / 256 : 1184);
            mark_ends_kernel<<<b2, 256, 0, st>>>(d_offsets, n_rec, total, reinterpret_cast<uint32_t *>(f->gmask), f->k, f->d_flag);
            CK(cudaGetLastError());
            g_launches++;
        }
        CK(f->entry->query(p, st));
        g_launches++;
        if (d_counts) {
            rc = run_count_records(d_bitmap, d_offsets, n_rec, total, d_counts, st, f->d_flag);
            if (rc) return rc;
        }
        return mark(f, 3, st);
    }
    rc = run_main<false>(f, total, d_bitmap, st);
    if (rc) return rc;
    rc = mark(f, 2, st);
    if (rc) return rc;
    if (d_counts && d_offsets && n_rec) {
        rc = run_count_records(d_bitmap, d_offsets, n_rec, total, d_counts, st);
        if (rc) return rc;
        rc = mark(f, 3, st);
    }
    return rc;
}

} // namespace

// =============================================================================================
// C ABI — device-facing
// =============================================================================================
extern "C" {

const char *sbf_last_error(void) { return g_err.c_str(); }
uint64_t sbf_kernel_launches(void) { return g_launches.load(); }

sbf_t *sbf_create(int k, int m, int s, int H, uint64_t num_bits) { return sbf_create_ex(k, m, s, H, num_bits, SBF_ALPHABET_DNA); }

sbf_t *sbf_create_ex(int k, int m, int s, int H, uint64_t num_bits, int alphabet)
{
    g_err.clear();
    const int sym_bits = alphabet == SBF_ALPHABET_DNA ? 2 : alphabet == SBF_ALPHABET_PROTEIN ? 5 : alphabet == SBF_ALPHABET_DNA_TRIPLET ? 6 : 0;
    if (!sym_bits) {
        fail(SBF_ERR_INVALID_ARG, "sbf_create_ex: unknown alphabet");
        return nullptr;
    }
    if (k < 1 || k * sym_bits > 128 || m < 1 || m > k || s < 1 || s > k || H < 1 || H > 32 || num_bits < 1) {
        fail(SBF_ERR_INVALID_ARG, "sbf_create: need 1<=k, k*symbol_bits<=128 (DNA k<=64, protein k<=25, triplets k<=21), 1<=m<=k, 1<=s<=k, 1<=H<=32, num_bits>=1");
        return nullptr;
    }
    uint64_t need = (num_bits + 255) / 256, shards = 1;
    int P = 0;
    while (shards < need) { shards <<= 1; ++P; } // rounded up to a power of two (A8)
    if (P > 32) {
        fail(SBF_ERR_UNSUPPORTED, "sbf_create: more than 2^32 shards");
        return nullptr;
    }
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        fail_cuda(e, "sbf_create: no CUDA device (this library has no CPU fallback)");
        return nullptr;
    }
    sbf *f = new (std::nothrow) sbf();
    if (!f) {
        fail(SBF_ERR_NOMEM, "sbf_create: host allocation failed");
        return nullptr;
    }
    f->k = k; f->m = m; f->s = s; f->H = H; f->P = P; f->device = dev;
    f->alphabet = alphabet; f->sym_bits = sym_bits; f->sym_bytes = alphabet == SBF_ALPHABET_DNA_TRIPLET ? 3 : 1;
    // DNA with 33 <= k <= 64 has specialised streaming instances too (folded wide windows, A21); without one: wide_tile_kernel
    // (with 2^32 shards the instances are not used at all — see f->entry below — and naive_kernel packs a k-mer into one
    // 64-bit word, so k > 32 must take the wide kernel there as well)
    f->wide = alphabet != SBF_ALPHABET_DNA || (k > 32 && (P >= 32 || find_entry(k, m, s, H) == nullptr));
    f->num_shards = shards;
    f->host_chunk = kHostChunkDefault;
    f->tma_flush = shards * 32 >= kTmaFlushMinBytes;
    f->entry = (P < 32 && !f->wide) ? find_entry(k, m, s, H) : nullptr; // the specialised kernels take sigma's shift as a multiply by 2^P
    e = cudaMalloc(&f->filter, shards * 32);
    if (e == cudaSuccess) e = cudaMemset(f->filter, 0, shards * 32);
    if (e == cudaSuccess) e = cudaMalloc(&f->d_flag, 256);
    if (e == cudaSuccess) e = cudaMalloc(&f->d_long, (size_t)kLongCap * sizeof(uint2));
    if (e != cudaSuccess) {
        fail_cuda(e, "sbf_create: filter allocation");
        if (f->filter) cudaFree(f->filter);
        if (f->d_flag) cudaFree(f->d_flag);
        if (f->d_long) cudaFree(f->d_long);
        delete f;
        return nullptr;
    }
    // a7: L2 persistence window when the whole filter fits the persisting carve-out
    int max_persist = 0, max_window = 0;
    cudaDeviceGetAttribute(&max_persist, cudaDevAttrMaxPersistingL2CacheSize, dev);
    cudaDeviceGetAttribute(&max_window, cudaDevAttrMaxAccessPolicyWindowSize, dev);
    uint64_t bytes = shards * 32;
    // opt-in since round 3 (SBF_L2_WINDOW=1): measured to buy nothing on config 2 (profiles/l2_window_r03.md), and it is the
    // only device-wide side effect sbf_create had
    const char *l2_env = getenv("SBF_L2_WINDOW");
    const bool l2_allowed = l2_env && l2_env[0] == '1';
    if (l2_allowed && max_persist > 0 && bytes <= (uint64_t)max_persist && bytes <= (uint64_t)max_window && bytes >= (1u << 20)) {
        size_t cur = 0;
        cudaDeviceGetLimit(&cur, cudaLimitPersistingL2CacheSize);
        if (cur < bytes) cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, (size_t)max_persist);
        f->l2_window = (cudaGetLastError() == cudaSuccess);
    }
    return f;
}

void sbf_destroy(sbf_t *f)
{
    if (!f) return;
    cudaDeviceSynchronize();
    delete f->host;
    delete f->fastx;
    for (int i = 0; i < 4; ++i)
        if (f->tev[i]) cudaEventDestroy(f->tev[i]);
    if (f->packed) cudaFree(f->packed);
    if (f->gmask) cudaFree(f->gmask);
    if (f->filter) cudaFree(f->filter);
    if (f->d_flag) cudaFree(f->d_flag);
    if (f->d_long) cudaFree(f->d_long);
    cudaGetLastError();
    delete f;
}

uint64_t sbf_num_bits(const sbf_t *f) { return f ? f->num_shards * 256 : 0; }
uint64_t sbf_num_shards(const sbf_t *f) { return f ? f->num_shards : 0; }
int sbf_is_specialized(const sbf_t *f) { return (f && f->entry) ? 1 : 0; }
const uint64_t *sbf_filter_device_ptr(const sbf_t *f) { return f ? f->filter : nullptr; }

int sbf_reserve(sbf_t *f, uint64_t max_bases)
{
    if (!f) return fail(SBF_ERR_INVALID_ARG, "sbf_reserve: NULL handle");
    return ensure_scratch(f, max_bases);
}

int sbf_set_host_chunk(sbf_t *f, uint64_t symbols)
{
    if (!f) return fail(SBF_ERR_INVALID_ARG, "sbf_set_host_chunk: NULL handle");
    if (symbols == 0 || (symbols & 127) || symbols < 128 + (uint64_t)f->k * (uint64_t)f->sym_bytes)
        return fail(SBF_ERR_INVALID_ARG, "sbf_set_host_chunk: need a multiple of 128 symbols, larger than k + 128");
    f->host_chunk = symbols;
    return SBF_OK;
}

int sbf_set_timing(sbf_t *f, int on)
{
    if (!f) return fail(SBF_ERR_INVALID_ARG, "sbf_set_timing: NULL handle");
    if (on)
        for (int i = 0; i < 4; ++i)
            if (!f->tev[i]) CK(cudaEventCreate(&f->tev[i]));
    f->timing = on != 0;
    f->tev_count = false;
    f->tev_valid = false;
    return SBF_OK;
}

int sbf_get_timing(sbf_t *f, float *ms3)
{
    if (!f || !ms3) return fail(SBF_ERR_INVALID_ARG, "sbf_get_timing: NULL argument");
    if (!f->timing) return fail(SBF_ERR_INVALID_ARG, "sbf_get_timing: timing is off (sbf_set_timing)");
    ms3[0] = ms3[1] = ms3[2] = 0.f;
    if (!f->tev_valid) return fail(SBF_ERR_INVALID_ARG, "sbf_get_timing: no timed call yet");
    CK(cudaEventSynchronize(f->tev[f->tev_count ? 3 : 2]));
    CK(cudaEventElapsedTime(&ms3[0], f->tev[0], f->tev[1]));
    CK(cudaEventElapsedTime(&ms3[1], f->tev[1], f->tev[2]));
    if (f->tev_count) CK(cudaEventElapsedTime(&ms3[2], f->tev[2], f->tev[3]));
    return SBF_OK;
}

int sbf_clear(sbf_t *f, void *stream)
{
    if (!f) return fail(SBF_ERR_INVALID_ARG, "sbf_clear: NULL handle");
    CK(cudaMemsetAsync(f->filter, 0, f->num_shards * 32, (cudaStream_t)stream));
    return SBF_OK;
}

int sbf_insert_seq(sbf_t *f, const char *d_seq, uint64_t len, void *stream)
{
    if (!f || (!d_seq && len)) return fail(SBF_ERR_INVALID_ARG, "sbf_insert_seq: NULL argument");
    return run_insert(f, d_seq, nullptr, 0, len, (cudaStream_t)stream);
}

int sbf_insert_records(sbf_t *f, const char *d_bases, const uint64_t *d_offsets, uint64_t n_rec, uint64_t total_bases,
                       void *stream)
{
    if (!f || (!d_bases && total_bases) || (!d_offsets && n_rec)) return fail(SBF_ERR_INVALID_ARG, "sbf_insert_records: NULL argument");
    if (n_rec == 0 && total_bases) return fail(SBF_ERR_INVALID_ARG, "sbf_insert_records: bases without records");
    return run_insert(f, d_bases, d_offsets, n_rec, total_bases, (cudaStream_t)stream);
}

int sbf_query_seq(sbf_t *f, const char *d_seq, uint64_t len, uint32_t *d_bitmap, uint64_t *d_hits, void *stream)
{
    if (!f || (!d_seq && len) || (!d_bitmap && len)) return fail(SBF_ERR_INVALID_ARG, "sbf_query_seq: NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    int rc = run_query(f, d_seq, nullptr, 0, len, d_bitmap, nullptr, st);
    if (rc) return rc;
    if (d_hits) {
        CK(cudaMemsetAsync(d_hits, 0, sizeof(uint64_t), st));
        uint64_t nw = (len + 31) / 32;
        if (nw) {
            unsigned blocks = (unsigned)((nw + 255) / 256 < 1184 ? (nw + 255) / 256 : 1184);
            count_total_kernel<<<blocks, 256, 0, st>>>(d_bitmap, nw, reinterpret_cast<unsigned long long *>(d_hits));
            CK(cudaGetLastError());
            g_launches++;
            rc = mark(f, 3, st);
            if (rc) return rc;
        }
    }
    return SBF_OK;
}

int sbf_query_records(sbf_t *f, const char *d_bases, const uint64_t *d_offsets, uint64_t n_rec, uint64_t total_bases,
                      uint32_t *d_bitmap, uint32_t *d_hit_counts, void *stream)
{
    if (!f || (!d_bases && total_bases) || (!d_offsets && n_rec) || (!d_bitmap && total_bases))
        return fail(SBF_ERR_INVALID_ARG, "sbf_query_records: NULL argument");
    if (n_rec == 0 && total_bases) return fail(SBF_ERR_INVALID_ARG, "sbf_query_records: bases without records");
    cudaStream_t st = (cudaStream_t)stream;
    if (d_hit_counts && n_rec && total_bases == 0) CK(cudaMemsetAsync(d_hit_counts, 0, n_rec * sizeof(uint32_t), st));
    return run_query(f, d_bases, d_offsets, n_rec, total_bases, d_bitmap, d_hit_counts, st);
}

int sbf_export_bits(const sbf_t *f, void *h_dst, uint64_t nbytes)
{
    if (!f || !h_dst) return fail(SBF_ERR_INVALID_ARG, "sbf_export_bits: NULL argument");
    if (nbytes != f->num_shards * 32) return fail(SBF_ERR_INVALID_ARG, "sbf_export_bits: nbytes must be 32*numShards");
    CK(cudaDeviceSynchronize());
    CK(cudaMemcpy(h_dst, f->filter, nbytes, cudaMemcpyDeviceToHost));
    return SBF_OK;
}

int sbf_import_bits(sbf_t *f, const void *h_src, uint64_t nbytes)
{
    if (!f || !h_src) return fail(SBF_ERR_INVALID_ARG, "sbf_import_bits: NULL argument");
    if (nbytes != f->num_shards * 32) return fail(SBF_ERR_INVALID_ARG, "sbf_import_bits: nbytes must be 32*numShards");
    CK(cudaDeviceSynchronize());
    CK(cudaMemcpy(f->filter, h_src, nbytes, cudaMemcpyHostToDevice));
    return SBF_OK;
}

int sbf_or_bits_device(sbf_t *f, const uint64_t *d_src, uint64_t nbytes, void *stream)
{
    if (!f || !d_src) return fail(SBF_ERR_INVALID_ARG, "sbf_or_bits_device: NULL argument");
    if (nbytes != f->num_shards * 32) return fail(SBF_ERR_INVALID_ARG, "sbf_or_bits_device: nbytes must be 32*numShards");
    uint64_t nw = f->num_shards * 4;
    unsigned blocks = (unsigned)((nw / 2 + 255) / 256 < 2368 ? (nw / 2 + 255) / 256 : 2368);
    or_words_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(f->filter, d_src, nw);
    CK(cudaGetLastError());
    g_launches++;
    return SBF_OK;
}

int sbf_or_range_device(sbf_t *f, uint64_t offset_bytes, const uint64_t *d_src, uint64_t nbytes, void *stream)
{
    if (!f || !d_src) return fail(SBF_ERR_INVALID_ARG, "sbf_or_range_device: NULL argument");
    if ((offset_bytes & 31) || (nbytes & 31) || offset_bytes + nbytes > f->num_shards * 32 ||
        (reinterpret_cast<uintptr_t>(d_src) & 15))
        return fail(SBF_ERR_INVALID_ARG, "sbf_or_range_device: range must be whole shards inside the filter, source 16-byte aligned");
    uint64_t nw = nbytes / 8;
    if (nw == 0) return SBF_OK;
    unsigned blocks = (unsigned)((nw / 2 + 255) / 256 < 2368 ? (nw / 2 + 255) / 256 : 2368);
    or_words_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(f->filter + offset_bytes / 8, d_src, nw);
    CK(cudaGetLastError());
    g_launches++;
    return SBF_OK;
}

int sbf_or_peers_range_device(sbf_t *f, uint64_t offset_bytes, const uint64_t *const *d_peer_ranges, int n_peers, uint64_t nbytes,
                              void *stream)
{
    if (!f || (!d_peer_ranges && n_peers)) return fail(SBF_ERR_INVALID_ARG, "sbf_or_peers_range_device: NULL argument");
    if (n_peers < 0 || n_peers > kMaxPeers) return fail(SBF_ERR_INVALID_ARG, "sbf_or_peers_range_device: at most 15 peers per call");
    if ((offset_bytes & 31) || (nbytes & 31) || offset_bytes + nbytes > f->num_shards * 32)
        return fail(SBF_ERR_INVALID_ARG, "sbf_or_peers_range_device: range must be whole shards inside the filter");
    PeerPtrs pp;
    for (int j = 0; j < kMaxPeers; ++j) pp.p[j] = nullptr;
    for (int j = 0; j < n_peers; ++j) {
        if (!d_peer_ranges[j] || (reinterpret_cast<uintptr_t>(d_peer_ranges[j]) & 15))
            return fail(SBF_ERR_INVALID_ARG, "sbf_or_peers_range_device: peer pointers must be non-NULL and 16-byte aligned");
        pp.p[j] = d_peer_ranges[j];
    }
    const uint64_t nw = nbytes / 8;
    if (nw == 0 || n_peers == 0) return SBF_OK;
    unsigned blocks = (unsigned)((nw / 2 + 255) / 256 < 2368 ? (nw / 2 + 255) / 256 : 2368);
    or_peers_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(f->filter + offset_bytes / 8, pp, n_peers, nw);
    CK(cudaGetLastError());
    g_launches++;
    return SBF_OK;
}

int sbf_ipc_export_filter(const sbf_t *f, void *handle64)
{
    if (!f || !handle64) return fail(SBF_ERR_INVALID_ARG, "sbf_ipc_export_filter: NULL argument");
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "cudaIpcMemHandle_t is 64 bytes");
    CK(cudaIpcGetMemHandle(reinterpret_cast<cudaIpcMemHandle_t *>(handle64), f->filter));
    return SBF_OK;
}

int sbf_ipc_open_filter(const void *handle64, uint64_t **d_ptr)
{
    if (!handle64 || !d_ptr) return fail(SBF_ERR_INVALID_ARG, "sbf_ipc_open_filter: NULL argument");
    cudaIpcMemHandle_t h;
    memcpy(&h, handle64, sizeof(h));
    void *p = nullptr;
    CK(cudaIpcOpenMemHandle(&p, h, cudaIpcMemLazyEnablePeerAccess));
    *d_ptr = static_cast<uint64_t *>(p);
    return SBF_OK;
}

int sbf_ipc_close_filter(uint64_t *d_ptr)
{
    if (!d_ptr) return SBF_OK;
    CK(cudaIpcCloseMemHandle(d_ptr));
    return SBF_OK;
}

} // extern "C"

// =============================================================================================
// C ABI — host-facing ("host-facing calls synchronise"; staging after P:323-325):
// the batch is cut in chunks of host_chunk symbols (default 32 Mi) that overlap by k-1, so that every k-mer
// start position belongs to exactly one chunk and is complete inside it.  A copy stream moves
// chunk c+1 to the device while the compute stream packs and walks chunk c; results come back
// chunk by chunk.  Pageable caller memory is staged through two pinned buffers; pinned or
// registered caller memory is copied from directly.
// =============================================================================================
namespace {


bool is_pinned(const void *p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeHost;
}

// insert (h_bitmap == nullptr) or query of a host-resident batch
int run_host(sbf *f, bool insert, const char *h_bases, const uint64_t *h_offsets, uint64_t n_rec, uint64_t total,
             uint32_t *h_bitmap, uint32_t *h_counts, uint64_t *h_hits)
{
    if (h_hits) *h_hits = 0;
    if (total == 0) {
        if (h_counts && n_rec) memset(h_counts, 0, n_rec * sizeof(uint32_t));
        return SBF_OK;
    }
    // the internal streams are non-blocking: order this call after everything the caller enqueued before it
    CK(cudaDeviceSynchronize());
    const uint64_t ov = (uint64_t)f->k * (uint64_t)f->sym_bytes - 1; // bytes a k-mer extends past its first one
    const uint64_t kHostChunk = f->host_chunk;
    const uint64_t span = (total < kHostChunk ? total : kHostChunk) + ov; // largest chunk incl. overlap
    const uint64_t n_chunks = (total + kHostChunk - 1) / kHostChunk;
    const bool direct = is_pinned(h_bases);
    // most record boundaries a chunk can hold: all of them (+2 ends).  Empty records repeat an offset, so the
    // chunk's symbol count is NOT a bound.
    const uint64_t max_off = h_offsets ? n_rec + 2 : 2;

    if (!f->host) {
        f->host = new (std::nothrow) HostRun();
        if (!f->host) return fail(SBF_ERR_NOMEM, "host staging: allocation failed");
        CK(cudaStreamCreateWithFlags(&f->host->copy, cudaStreamNonBlocking));
        CK(cudaStreamCreateWithFlags(&f->host->comp, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CK(cudaEventCreateWithFlags(&f->host->copied[i], cudaEventDisableTiming));
            CK(cudaEventCreateWithFlags(&f->host->computed[i], cudaEventDisableTiming));
        }
        CK(cudaEventCreateWithFlags(&f->host->offs_ready, cudaEventDisableTiming));
    }
    HostRun &R = *f->host;
    const int slots = n_chunks > 1 ? 2 : 1;
    if (R.cap_bases < span) { // grow the device symbol slots (both, so a later multi-chunk call finds them)
        for (int i = 0; i < 2; ++i) {
            if (R.d_bases[i]) cudaFree(R.d_bases[i]);
            R.d_bases[i] = nullptr;
        }
        R.cap_bases = 0;
        for (int i = 0; i < 2; ++i) CK(cudaMalloc(&R.d_bases[i], span + 16));
        R.cap_bases = span;
    }
    if (!direct && R.cap_pin < span) {
        for (int i = 0; i < 2; ++i) {
            if (R.pin[i]) cudaFreeHost(R.pin[i]);
            R.pin[i] = nullptr;
        }
        R.cap_pin = 0;
        for (int i = 0; i < 2; ++i) CK(cudaMallocHost(&R.pin[i], span));
        R.cap_pin = span;
    }
    if (h_offsets && R.cap_off < max_off) {
        for (int i = 0; i < 2; ++i) {
            if (R.d_off[i]) cudaFree(R.d_off[i]);
            R.d_off[i] = nullptr;
        }
        R.cap_off = 0;
        for (int i = 0; i < 2; ++i) CK(cudaMalloc(&R.d_off[i], max_off * sizeof(uint64_t)));
        R.cap_off = max_off;
    }
    if (h_offsets) { // the batch's offsets go to the device ONCE; every chunk's own offsets are derived from them there
        if (R.cap_rec < n_rec + 1) {
            if (R.d_off_full) cudaFree(R.d_off_full);
            if (R.d_counts) cudaFree(R.d_counts);
            R.d_off_full = nullptr; R.d_counts = nullptr; R.cap_rec = 0;
            CK(cudaMalloc(&R.d_off_full, (n_rec + 1) * sizeof(uint64_t)));
            CK(cudaMalloc(&R.d_counts, (n_rec + 1) * sizeof(uint32_t)));
            R.cap_rec = n_rec + 1;
        }
        CK(cudaMemcpyAsync(R.d_off_full, h_offsets, (n_rec + 1) * sizeof(uint64_t), cudaMemcpyHostToDevice, R.copy));
        CK(cudaEventRecord(R.offs_ready, R.copy));
        CK(cudaStreamWaitEvent(R.comp, R.offs_ready, 0));
    }
    (void)slots;
    const uint64_t n_bm = (total + 31) / 32;
    if (!insert) {
        if (R.cap_bitmap < n_bm + 4) {
            if (R.d_bitmap) cudaFree(R.d_bitmap);
            R.d_bitmap = nullptr; R.cap_bitmap = 0;
            CK(cudaMalloc(&R.d_bitmap, (n_bm + 4) * sizeof(uint32_t)));
            R.cap_bitmap = n_bm + 4;
        }
        if (h_hits && !R.d_hits) CK(cudaMalloc(&R.d_hits, sizeof(unsigned long long)));
    }
    int rc = ensure_scratch(f, span);
    if (rc) return rc;

    uint64_t off_lo = 0; // first offset index with h_offsets[i] > chunk start (monotone over chunks)
    for (uint64_t c = 0; c < n_chunks; ++c) {
        const int sl = (int)(c & 1);
        const uint64_t a = c * kHostChunk;
        const uint64_t e = (a + kHostChunk + ov < total) ? a + kHostChunk + ov : total;
        const uint64_t n = e - a;
        if (c >= 2) {
            CK(cudaEventSynchronize(R.copied[sl]));                 // pinned slot free again
            CK(cudaStreamWaitEvent(R.copy, R.computed[sl], 0));     // device slot free again
        }
        uint64_t n_off = 0;
        if (h_offsets) {
            // record boundaries strictly inside (a, e): indices [lo, hi) of the batch's offsets
            const uint64_t *lo = std::upper_bound(h_offsets + off_lo, h_offsets + n_rec + 1, a);
            const uint64_t *hi = std::lower_bound(lo, h_offsets + n_rec + 1, e);
            off_lo = (uint64_t)(lo - h_offsets);
            f->phase0 = (int)((a - *(lo - 1)) % (uint64_t)f->sym_bytes); // triplets: the chunk's first record started at *(lo-1)
            const uint64_t n_inner = (uint64_t)(hi - lo);
            n_off = n_inner + 2;
            rebase_offsets_kernel<<<(unsigned)((n_inner + 256) / 256), 256, 0, R.comp>>>(R.d_off_full + off_lo, n_inner, a, n,
                                                                                       R.d_off[sl]);
            CK(cudaGetLastError());
            g_launches++;
        }
        if (!h_offsets) f->phase0 = (int)(a % (uint64_t)f->sym_bytes);
        const char *src = h_bases + a;
        if (!direct) {
            memcpy(R.pin[sl], src, n);
            src = R.pin[sl];
        }
        CK(cudaMemcpyAsync(R.d_bases[sl], src, n, cudaMemcpyHostToDevice, R.copy));
        CK(cudaEventRecord(R.copied[sl], R.copy));
        CK(cudaStreamWaitEvent(R.comp, R.copied[sl], 0));
        const uint64_t *d_off = h_offsets ? R.d_off[sl] : nullptr;
        const uint64_t nr = h_offsets ? n_off - 1 : 0;
        if (insert) {
            rc = run_insert(f, R.d_bases[sl], d_off, nr, n, R.comp);
        } else {
            rc = run_query(f, R.d_bases[sl], d_off, nr, n, R.d_bitmap + a / 32, nullptr, R.comp);
        }
        f->phase0 = 0;
        if (rc) return rc;
        CK(cudaEventRecord(R.computed[sl], R.comp));
        if (!insert && h_bitmap) {
            const uint64_t w0 = a / 32;
            const uint64_t w1 = (c + 1 == n_chunks) ? n_bm : (a + kHostChunk) / 32;
            CK(cudaMemcpyAsync(h_bitmap + w0, R.d_bitmap + w0, (w1 - w0) * sizeof(uint32_t), cudaMemcpyDeviceToHost, R.comp));
        }
    }
    if (!insert) {
        CK(cudaStreamSynchronize(R.copy));
        if (h_counts && n_rec) {
            rc = run_count_records(R.d_bitmap, R.d_off_full, n_rec, total, R.d_counts, R.comp);
            if (rc) return rc;
            CK(cudaMemcpyAsync(h_counts, R.d_counts, n_rec * sizeof(uint32_t), cudaMemcpyDeviceToHost, R.comp));
        }
        if (h_hits) {
            CK(cudaMemsetAsync(R.d_hits, 0, sizeof(unsigned long long), R.comp));
            unsigned blocks = (unsigned)((n_bm + 255) / 256 < 1184 ? (n_bm + 255) / 256 : 1184);
            count_total_kernel<<<blocks, 256, 0, R.comp>>>(R.d_bitmap, n_bm, R.d_hits);
            CK(cudaGetLastError());
            g_launches++;
            CK(cudaMemcpyAsync(h_hits, R.d_hits, sizeof(uint64_t), cudaMemcpyDeviceToHost, R.comp));
        }
    }
    CK(cudaStreamSynchronize(R.copy));
    CK(cudaStreamSynchronize(R.comp));
    return SBF_OK;
}

} // namespace

extern "C" {

int sbf_insert_seq_host(sbf_t *f, const char *h_seq, uint64_t len)
{
    if (!f || (!h_seq && len)) return fail(SBF_ERR_INVALID_ARG, "sbf_insert_seq_host: NULL argument");
    return run_host(f, true, h_seq, nullptr, 0, len, nullptr, nullptr, nullptr);
}

int sbf_insert_records_host(sbf_t *f, const char *h_bases, const uint64_t *h_offsets, uint64_t n_rec)
{
    if (!f || !h_offsets) return fail(SBF_ERR_INVALID_ARG, "sbf_insert_records_host: NULL argument");
    uint64_t total = h_offsets[n_rec];
    if (!h_bases && total) return fail(SBF_ERR_INVALID_ARG, "sbf_insert_records_host: NULL bases");
    return run_host(f, true, h_bases, h_offsets, n_rec, total, nullptr, nullptr, nullptr);
}

int sbf_query_seq_host(sbf_t *f, const char *h_seq, uint64_t len, uint32_t *h_bitmap, uint64_t *h_hits)
{
    if (!f || (!h_seq && len) || (!h_bitmap && len)) return fail(SBF_ERR_INVALID_ARG, "sbf_query_seq_host: NULL argument");
    return run_host(f, false, h_seq, nullptr, 0, len, h_bitmap, nullptr, h_hits);
}

int sbf_query_records_host(sbf_t *f, const char *h_bases, const uint64_t *h_offsets, uint64_t n_rec, uint32_t *h_bitmap,
                           uint32_t *h_hit_counts)
{
    if (!f || !h_offsets) return fail(SBF_ERR_INVALID_ARG, "sbf_query_records_host: NULL argument");
    uint64_t total = h_offsets[n_rec];
    if ((!h_bases || !h_bitmap) && total) return fail(SBF_ERR_INVALID_ARG, "sbf_query_records_host: NULL buffer");
    return run_host(f, false, h_bases, h_offsets, n_rec, total, h_bitmap, h_hit_counts, nullptr);
}

} // extern "C"

// =============================================================================================
// C ABI — FASTA / FASTQ text in host memory ("streamed FASTA/FASTQ input"; "Host FASTX staging").
// The raw text is cut in chunks of host_chunk bytes; a copy stream moves chunk c+1 to the device while the compute
// stream normalises chunk c there (sbf_fastx.cuh: headers, quality lines and line ends dropped, sequence bytes
// compacted into a dense record batch + offsets) and runs the ordinary record-batch insert / query on it.  The lexer
// state and the last k-1 bytes of the open record travel from chunk to chunk in device memory; the host reads back
// 24 bytes per chunk (the batch's size), which is what it needs to size the launches.
// =============================================================================================
namespace {

template <int FMT>
int fastx_normalise_chunk(FastxRun &R, int sl, uint64_t n, const FastxState *st, FastxState *st_next, uint32_t keep, bool last)
{
    const uint32_t n_tiles = (uint32_t)((n + kFxTile - 1) / kFxTile);
    if (n_tiles) {
        fastx_tile_kernel<FMT><<<n_tiles, kFxThreads, 0, R.comp>>>(R.d_text[sl], n, st, R.d_tiles);
        CK(cudaGetLastError());
    }
    fastx_scan_kernel<FMT><<<1, 32, 0, R.comp>>>(R.d_tiles, n_tiles, R.d_text[sl], n, const_cast<FastxState *>(st), st_next, R.d_off[sl]);
    CK(cudaGetLastError());
    if (n_tiles) {
        fastx_emit_kernel<FMT><<<n_tiles, kFxThreads, 0, R.comp>>>(R.d_text[sl], n, st, R.d_tiles, R.d_dense[sl], R.d_off[sl]);
        CK(cudaGetLastError());
    }
    g_launches += n_tiles ? 3 : 1;
    if (!last) {
        fastx_carry_kernel<<<1, 64, 0, R.comp>>>(R.d_dense[sl], R.d_off[sl], st, keep, R.d_dense[sl ^ 1], st_next);
        CK(cudaGetLastError());
        g_launches++;
    }
    return SBF_OK;
}

int run_fastx(sbf *f, bool insert, const char *h_text, uint64_t n_bytes, int format, uint32_t *h_counts, uint64_t max_records,
              uint64_t *out_records, uint64_t *out_bases)
{
    if (out_records) *out_records = 0;
    if (out_bases) *out_bases = 0;
    if (format == 0) { // detect from the first byte that is not white space
        uint64_t i = 0;
        while (i < n_bytes && (h_text[i] == '\n' || h_text[i] == '\r' || h_text[i] == ' ')) ++i;
        format = (i < n_bytes && h_text[i] == '@') ? kFxFastq : kFxFasta;
    }
    if (format != kFxFasta && format != kFxFastq) return fail(SBF_ERR_INVALID_ARG, "fastx: format must be 0 (detect), 1 (FASTA) or 2 (FASTQ)");
    if (n_bytes == 0) return SBF_OK;
    CK(cudaDeviceSynchronize()); // order this call after everything enqueued before it (the internal streams are non-blocking)
    const uint64_t chunk = f->host_chunk;
    const uint64_t n_chunks = (n_bytes + chunk - 1) / chunk;
    const uint32_t keep = (uint32_t)(f->k * f->sym_bytes - 1);
    const uint64_t span = (n_bytes < chunk ? n_bytes : chunk);
    if (!f->fastx) {
        f->fastx = new (std::nothrow) FastxRun();
        if (!f->fastx) return fail(SBF_ERR_NOMEM, "fastx: allocation failed");
        FastxRun &N = *f->fastx;
        CK(cudaStreamCreateWithFlags(&N.copy, cudaStreamNonBlocking));
        CK(cudaStreamCreateWithFlags(&N.comp, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CK(cudaEventCreateWithFlags(&N.copied[i], cudaEventDisableTiming));
            CK(cudaEventCreateWithFlags(&N.computed[i], cudaEventDisableTiming));
        }
        CK(cudaEventCreateWithFlags(&N.normalised, cudaEventDisableTiming));
        CK(cudaMalloc(&N.d_state, 2 * sizeof(FastxState)));
        CK(cudaMallocHost(&N.h_state, sizeof(FastxState)));
    }
    FastxRun &R = *f->fastx;
    const bool direct = is_pinned(h_text);
    if (R.cap_text < span) { // every buffer below is sized by the text bytes of one chunk
        for (int i = 0; i < 2; ++i) {
            if (R.pin[i]) cudaFreeHost(R.pin[i]);
            if (R.d_text[i]) cudaFree(R.d_text[i]);
            if (R.d_dense[i]) cudaFree(R.d_dense[i]);
            if (R.d_off[i]) cudaFree(R.d_off[i]);
            R.pin[i] = nullptr; R.d_text[i] = nullptr; R.d_dense[i] = nullptr; R.d_off[i] = nullptr;
        }
        if (R.d_tiles) cudaFree(R.d_tiles);
        if (R.d_bitmap) cudaFree(R.d_bitmap);
        if (R.d_counts_local) cudaFree(R.d_counts_local);
        R.d_tiles = nullptr; R.d_bitmap = nullptr; R.d_counts_local = nullptr; R.cap_text = 0;
        const uint64_t max_rec = span / 2 + 3; // a record start needs ">" and a line end before the next one
        for (int i = 0; i < 2; ++i) {
            CK(cudaMallocHost(&R.pin[i], span));
            CK(cudaMalloc(&R.d_text[i], span + 16));
            CK(cudaMalloc(&R.d_dense[i], span + keep + 64));
            CK(cudaMalloc(&R.d_off[i], (max_rec + 2) * sizeof(uint64_t)));
        }
        CK(cudaMalloc(&R.d_tiles, ((span + kFxTile - 1) / kFxTile + 1) * sizeof(Seg)));
        CK(cudaMalloc(&R.d_bitmap, ((span + keep + 64 + 31) / 32 + 4) * sizeof(uint32_t)));
        CK(cudaMalloc(&R.d_counts_local, (max_rec + 2) * sizeof(uint32_t)));
        R.cap_text = span;
    }
    if (!insert && h_counts && max_records) {
        if (R.cap_counts < max_records) {
            if (R.d_counts) cudaFree(R.d_counts);
            R.d_counts = nullptr; R.cap_counts = 0;
            CK(cudaMalloc(&R.d_counts, max_records * sizeof(uint32_t)));
            R.cap_counts = max_records;
        }
        CK(cudaMemsetAsync(R.d_counts, 0, max_records * sizeof(uint32_t), R.comp));
    }
    int rc = ensure_scratch(f, span + keep + 64);
    if (rc) return rc;
    FastxState init;
    memset(&init, 0, sizeof(init));
    init.at_line_start = 1;
    CK(cudaMemcpyAsync(&R.d_state[0], &init, sizeof(init), cudaMemcpyHostToDevice, R.comp));

    uint64_t rec_base = 0, bases_total = 0; // record starts / distinct sequence bytes before the current chunk
    uint32_t rec_prefix = 0;                // triplets: bytes of local record 0 that precede the dense buffer, mod 3
    for (uint64_t c = 0; c < n_chunks; ++c) {
        const int sl = (int)(c & 1);
        const uint64_t a = c * chunk;
        const uint64_t n = (a + chunk < n_bytes) ? chunk : n_bytes - a;
        if (c >= 2) {
            CK(cudaEventSynchronize(R.copied[sl]));
            CK(cudaStreamWaitEvent(R.copy, R.computed[sl], 0));
        }
        const char *src = h_text + a;
        if (!direct) {
            memcpy(R.pin[sl], src, n);
            src = R.pin[sl];
        }
        CK(cudaMemcpyAsync(R.d_text[sl], src, n, cudaMemcpyHostToDevice, R.copy));
        CK(cudaEventRecord(R.copied[sl], R.copy));
        CK(cudaStreamWaitEvent(R.comp, R.copied[sl], 0));
        FastxState *st = &R.d_state[c & 1], *st_next = &R.d_state[(c + 1) & 1];
        const bool last = c + 1 == n_chunks;
        rc = format == kFxFasta ? fastx_normalise_chunk<kFxFasta>(R, sl, n, st, st_next, keep, last)
                                : fastx_normalise_chunk<kFxFastq>(R, sl, n, st, st_next, keep, last);
        if (rc) return rc;
        CK(cudaMemcpyAsync(R.h_state, st, sizeof(FastxState), cudaMemcpyDeviceToHost, R.comp));
        CK(cudaEventRecord(R.normalised, R.comp));
        CK(cudaEventSynchronize(R.normalised)); // 40 bytes: the batch's size, needed to size the launches below
        const uint64_t n_bases = R.h_state->n_bases, n_starts = R.h_state->n_starts, carry = R.h_state->carry_len;
        const uint64_t n_rec = n_starts + 1;
        if (!insert && h_counts && rec_base + n_starts > max_records)
            return fail(SBF_ERR_INVALID_ARG, "sbf_query_fastx_host: more records in the text than max_records");
        f->phase0 = (int)(rec_prefix % (uint32_t)f->sym_bytes);
        if (n_bases) {
            if (insert) {
                rc = run_insert(f, reinterpret_cast<const char *>(R.d_dense[sl]), R.d_off[sl], n_rec, n_bases, R.comp);
            } else {
                rc = run_query(f, reinterpret_cast<const char *>(R.d_dense[sl]), R.d_off[sl], n_rec, n_bases, R.d_bitmap,
                               h_counts ? R.d_counts_local : nullptr, R.comp);
                if (!rc && h_counts) {
                    unsigned blocks = (unsigned)((n_rec + 255) / 256 < 1184 ? (n_rec + 255) / 256 : 1184);
                    fastx_add_counts_kernel<<<blocks, 256, 0, R.comp>>>(R.d_counts_local, n_rec, rec_base, R.d_counts, max_records);
                    rc = cudaGetLastError() == cudaSuccess ? SBF_OK : fail(SBF_ERR_CUDA, "fastx_add_counts_kernel");
                    g_launches++;
                }
            }
        }
        f->phase0 = 0;
        if (rc) return rc;
        CK(cudaEventRecord(R.computed[sl], R.comp));
        // the record that is open at the end of this chunk: how many of its bytes the next dense buffer will NOT hold
        // (host mirror of fastx_carry_kernel's choice; needs the last record's length, which the offsets hold on the
        // device — read back only for multi-byte symbols, where the 3-byte grid must survive the chunk edge)
        if (!last && f->sym_bytes > 1) {
            uint64_t last_start = 0;
            CK(cudaMemcpyAsync(&last_start, R.d_off[sl] + n_starts, sizeof(uint64_t), cudaMemcpyDeviceToHost, R.comp));
            CK(cudaStreamSynchronize(R.comp));
            const uint64_t len = n_bases - last_start;
            const uint64_t cl = len < keep ? len : keep;
            rec_prefix = (uint32_t)(((n_starts ? 0 : rec_prefix) + len - cl) % 3);
        }
        rec_base += n_starts;
        bases_total += n_bases - carry;
    }
    if (!insert && h_counts && rec_base)
        CK(cudaMemcpyAsync(h_counts, R.d_counts, rec_base * sizeof(uint32_t), cudaMemcpyDeviceToHost, R.comp));
    CK(cudaStreamSynchronize(R.copy));
    CK(cudaStreamSynchronize(R.comp));
    if (out_records) *out_records = rec_base;
    if (out_bases) *out_bases = bases_total;
    return SBF_OK;
}

} // namespace

extern "C" {

int sbf_insert_fastx_host(sbf_t *f, const char *h_text, uint64_t n_bytes, int format, uint64_t *n_records, uint64_t *n_bases)
{
    if (!f || (!h_text && n_bytes)) return fail(SBF_ERR_INVALID_ARG, "sbf_insert_fastx_host: NULL argument");
    return run_fastx(f, true, h_text, n_bytes, format, nullptr, 0, n_records, n_bases);
}

int sbf_query_fastx_host(sbf_t *f, const char *h_text, uint64_t n_bytes, int format, uint32_t *h_hit_counts, uint64_t max_records,
                         uint64_t *n_records, uint64_t *n_bases)
{
    if (!f || (!h_text && n_bytes)) return fail(SBF_ERR_INVALID_ARG, "sbf_query_fastx_host: NULL argument");
    return run_fastx(f, false, h_text, n_bytes, format, h_hit_counts, h_hit_counts ? max_records : 0, n_records, n_bases);
}

} // extern "C"

// =============================================================================================
// sbf_query_seq_static (include/sbf.h): the sequence query for callers that may not allocate device memory.
// Same two launches as sbf_query_seq on a handle — pack_kernel, then the chunk-mode query kernel — but the packed
// words and the validity mask go to an array that is part of the library image instead of cudaMalloc'ed scratch.
// =============================================================================================
namespace {
constexpr uint64_t kStaticMaxSymbols = SBF_STATIC_MAX_SYMBOLS;
constexpr uint64_t kStaticWords = (kStaticMaxSymbols + 15) / 16 + kPadWords;             // what pack_kernel writes at the limit
constexpr uint64_t kStaticPackedBytes = (kStaticWords * sizeof(uint32_t) + 255) / 256 * 256;
constexpr uint64_t kStaticMaskBytes = (kStaticWords * sizeof(uint16_t) + 8 + 255) / 256 * 256; // + 8 as ensure_scratch: the last mask store is 4 bytes wide
constexpr uint64_t kStaticBytes = kStaticPackedBytes + kStaticMaskBytes;                   // 6 MiB + 512 B
} // namespace

// The working memory itself: [0, kStaticPackedBytes) packed words, then the mask.  Every device that loads this
// module holds one copy until the process exits.  In host code this name is only a handle for the runtime's symbol
// table — never a device address, so it is never passed to a kernel; static_scratch() below asks the runtime
// where the current device keeps its copy.
static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

namespace {

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
unsigned char *g_static_ptr[kStaticMaxDevices]; // device address of g_static_scratch on device i, once looked up

// Device address of the array on the CURRENT device.  First call per device: one cudaGetSymbolAddress (it allocates
// nothing — the array came with the module — but it may make the runtime finish loading the module, which is why the
// header asks for the first call outside stream capture).  Later calls: a table read.
int static_scratch(unsigned char **out)
{
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices)
        return fail(SBF_ERR_UNSUPPORTED, "sbf_query_seq_static: device ordinal above 63");
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (g_static_ptr[dev] == nullptr) {
        void *p = nullptr;
        CK(cudaGetSymbolAddress(&p, g_static_scratch));
        if (p == nullptr) return fail(SBF_ERR_CUDA, "sbf_query_seq_static: the runtime returned no address for the static scratch array");
        g_static_ptr[dev] = static_cast<unsigned char *>(p);
    }
    *out = g_static_ptr[dev];
    return SBF_OK;
}

} // namespace

extern "C" {

int sbf_query_seq_static(int k, int m, int s, int H, const uint64_t *d_filter, uint64_t num_shards, const char *d_seq,
                         uint64_t len, uint32_t *d_bitmap, void *stream)
{
    if (k < 1 || k > 64 || m < 1 || m > k || s < 1 || s > k || H < 1 || H > 32)
        return fail(SBF_ERR_INVALID_ARG, "sbf_query_seq_static: need 1<=k<=64, 1<=m<=k, 1<=s<=k, 1<=H<=32");
    if (num_shards == 0 || (num_shards & (num_shards - 1)) != 0 || num_shards > (1ull << 32))
        return fail(SBF_ERR_INVALID_ARG, "sbf_query_seq_static: num_shards must be a power of two, at most 2^32");
    if (!d_filter || (reinterpret_cast<uintptr_t>(d_filter) & 31) != 0)
        return fail(SBF_ERR_INVALID_ARG, "sbf_query_seq_static: d_filter is NULL or not 32-byte aligned");
    if ((!d_seq && len) || (!d_bitmap && len)) return fail(SBF_ERR_INVALID_ARG, "sbf_query_seq_static: NULL argument");
    if (len > kStaticMaxSymbols) {
        char msg[224];
        snprintf(msg, sizeof(msg),
                 "sbf_query_seq_static: len = %llu symbols is above the static scratch limit SBF_STATIC_MAX_SYMBOLS = %llu; "
                 "split the sequence into pieces that overlap by k-1 symbols",
                 (unsigned long long)len, (unsigned long long)kStaticMaxSymbols);
        return fail(SBF_ERR_INVALID_ARG, msg);
    }
    int P = 0;
    while ((1ull << P) < num_shards) ++P;
    // same routing as sbf_create: a compiled instance where there is one (they take sigma's shift as a multiply by
    // 2^P, hence P < 32), else the runtime-parameter kernel, which packs a k-mer into one 64-bit word
    const KernelEntry *entry = P < 32 ? find_entry(k, m, s, H) : nullptr;
    if (entry == nullptr && k > 32)
        return fail(SBF_ERR_UNSUPPORTED, "sbf_query_seq_static: no streaming instance for this k > 32 (or 2^32 shards); use a handle");

    // set-up comes before the len == 0 exit so that an empty call at start-up does it
    unsigned char *scratch = nullptr;
    int rc = static_scratch(&scratch);
    if (rc) return rc;
    if (len == 0) return SBF_OK;

    cudaStream_t st = (cudaStream_t)stream;
    uint32_t *packed = reinterpret_cast<uint32_t *>(scratch);
    uint16_t *vmask = reinterpret_cast<uint16_t *>(scratch + kStaticPackedBytes);
    // a1: every word the query kernel will read (the pad words included) is rewritten here, so what the previous call
    // left in the array never reaches a result
    const uint64_t nw = (len + 15) / 16 + kPadWords;
    const unsigned pack_blocks = (unsigned)(((nw + 1) / 2 + 255) / 256);
    const int aligned = ((reinterpret_cast<uintptr_t>(d_seq) & 15) == 0) ? 1 : 0;
    pack_kernel<<<pack_blocks, 256, 0, st>>>(reinterpret_cast<const uint8_t *>(d_seq), len, packed, vmask, nw, k, aligned, nullptr,
                                             (len + 31) / 32, nullptr);
    CK(cudaGetLastError());
    g_launches++;

    // a2-a6: chunk-mode query, parameters as make_params() sets them for a handle
    StreamParams p;
    p.packed = packed;
    p.vmask = vmask;
    p.n_pos = len;
    p.filter = const_cast<uint64_t *>(d_filter); // the query kernels only load from it
    p.shard_shift = 32 - P;
    p.bitmap = d_bitmap;
    p.n_bitmap_words = (len + 31) / 32;
    p.chunk_blocks = len >= (64ull << 20) ? 8 : len >= (16ull << 20) ? 4 : 2;
    p.offsets = nullptr; p.n_rec = 0; p.counts = nullptr; p.fallback = nullptr; p.rec_limit = 0;
    p.long_groups = nullptr; p.long_cap = 0;
    if (entry) {
        CK(entry->query(p, st));
    } else {
        NaiveParams np;
        np.sp = p; np.k = k; np.m = m; np.s = s; np.H = H;
        const uint64_t n32 = (len + 31) / 32 * 32;
        naive_kernel<false><<<(unsigned)((n32 + 255) / 256), 256, 0, st>>>(np);
        CK(cudaGetLastError());
    }
    g_launches++;
    return SBF_OK;
}

} // extern "C"

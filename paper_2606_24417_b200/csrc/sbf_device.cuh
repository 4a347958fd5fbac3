// sbf_device.cuh — device code of the Super Bloom filter hot path (sm_100a).
//
// P:<n> = line n of the paper's extracted text; A<n> = reading n in DESIGN.md §3.
// This file restates the pinned arithmetic on its own; it shares nothing with oracle/.
//
// Kernels
//   pack_kernel        a1  ASCII -> 2-bit words (16 bases / uint32, first base in the top bits)
//                          + V, one bit per base: "no valid k-mer starts here" (a non-ACGT symbol among the
//                          next k, or fewer than k symbols left)
//   mark_ends_kernel   a1  chunk mode over records: ORs into V the k-1 start positions before every record
//                          end (a k-mer never spans two records)
//   stream_kernel      a2-a6  the fused, thread-serial streaming insert / query kernel (chunk mode)
//   stream_rec_kernel  a2-a6  the same query pipeline, one thread per short record (record mode)
//                          query test: SlidingGather (byte-gather form, H <= 4) or SlidingOr (256-bit masks)
//   stream_long_kernel a2-a6  the records of a record-mode batch that are too long for one thread, chunk by chunk
//   naive_kernel       a2-a6  runtime-parameter one-k-mer-per-thread form of Alg. 1/2 (any legal k,m,s,H)
//   wide_tile_kernel   a1-a6  the other alphabets and DNA k > 32 without an instance, from the ASCII bytes,
//                          runtime parameters, a tile of 1024 byte positions per CTA through shared memory
//   count kernels      a6  per-record / total popcount of the result bitmap
#pragma once

#include <cstdint>
#include <cuda_runtime.h>
#include <type_traits>
#include <utility>

// ---- tuning switches (defaults = the measured best)
#ifndef SBF_MINB_R
#define SBF_MINB_R 4 // record-mode query: 4 x 128 threads -> 128 registers
#endif
#ifndef SBF_Q_LA
#define SBF_Q_LA 7   // query: the minimizer runs this many positions ahead of the bit tests (1, 3, 7: 7 measured best)
#endif
#ifndef SBF_IDP_EXTRACT
#define SBF_IDP_EXTRACT 1 // bit-slice extraction by IDP.4A where the slice is byte aligned (H = 1, 2, 4, 8)
#endif
#ifndef SBF_FMA_ONEHOT
#define SBF_FMA_ONEHOT 0  // one-hot masks with one alu shift + three fma-pipe multiplies instead of two alu shifts (measured slower: more instructions)
#endif
#ifndef SBF_FMA_SIGMA
#define SBF_FMA_SIGMA 0   // sigma's final shift as a multiply-high by 2^P (fma pipe; measured: no gain)
#endif
#ifndef SBF_CPASYNC_L2_64B
#define SBF_CPASYNC_L2_64B 1 // query staging: cp.async with the .L2::64B prefetch-size hint (a miss then pulls 64 B from DRAM instead of 128 B: measured DRAM reads -44 %, same time)
#endif
#ifndef SBF_EARLY_RELOAD
#define SBF_EARLY_RELOAD 0 // query: reload the shard registers at the top of a step (measured: no gain, the scheduler already hides the LDS)
#endif
#ifndef SBF_PRED_RELOAD
#define SBF_PRED_RELOAD 1 // query: reload the shard registers with two predicated LDS.128 instead of a divergent branch
#endif
#ifndef SBF_GATHER
#define SBF_GATHER 1 // query: byte-gather sliding test (SlidingGather) instead of 256-bit masks where it applies (H <= 4, k-s+1 in {1,2,4,8})
#endif
#ifndef SBF_MIN3_ASM
#define SBF_MIN3_ASM 1 // sliding minimum: three-input minima as opaque asm (kept as VIMNMX3 instead of being re-associated)
#endif
#ifndef SBF_GATHER_PAIRED
#define SBF_GATHER_PAIRED 1 // SlidingGather, H = 4: the selectors of words q, q+1 share a register (one shift + one insert for both)
#endif
#ifndef SBF_GATHER_FMA_SHIFT
#define SBF_GATHER_FMA_SHIFT 0 // SlidingGather: right shifts of the y fields as multiply-high (fma pipe)
#endif
#ifndef SBF_MINB_I
#define SBF_MINB_I 5 // insert: CTAs per SM the register budget is cut for (5 x 128 threads -> 96 registers)
#endif
#ifndef SBF_MINB_Q
#define SBF_MINB_Q 5 // chunk-mode query, byte-gather form: 5 x 128 threads -> 96 registers (0.632 vs 0.640 ms per 240 Mbp at 4 CTAs); the mask form and the wider windows of k > 32 spill at 96 and stay at 4 x 128 threads -> 128 registers
#endif

namespace sbfk {

// ---- pinned constants (A1, A2, A4, A6) -------------------------------------------------
constexpr uint64_t kSeedM = 0x5851F42D4C957F2Dull;
constexpr uint32_t kMultG = 0x9E3779B1u;
constexpr uint64_t kGold64 = 0x9E3779B97F4A7C15ull;
constexpr uint64_t kSeedS = 0x2545F4914F6CDD1Dull;
constexpr uint64_t kMultF = 0xD6E8FEB86659FD93ull;

// ---- launch geometry ---------------------------------------------------------------------
constexpr int kChunk = 128;     // most k-mer start positions walked by one thread of stream_kernel (StreamParams::chunk_blocks * 16)
#ifndef SBF_STREAM_TPB
#define SBF_STREAM_TPB 128
#endif
constexpr int kStreamTPB = SBF_STREAM_TPB; // threads per CTA of stream_kernel
#ifndef SBF_REC_TPB
#define SBF_REC_TPB 128
#endif
constexpr int kRecTPB = SBF_REC_TPB; // threads per CTA of stream_rec_kernel
constexpr int kPadWords = 16;   // zero / all-invalid words appended to the packed sequence and its mask

struct StreamParams {
    const uint32_t *packed; // 2-bit words, ceil(n_pos/16) + kPadWords
    const uint16_t *vmask;  // one uint16 per packed word: bit j = V[16*word + j], "no valid k-mer starts at that symbol"
    uint64_t n_pos;         // symbols in the batch (= k-mer start positions walked)
    uint64_t *filter;       // 4 * numShards sector words
    int shard_shift;        // 32 - P
    uint32_t *bitmap;       // query: ceil(n_pos/32) words
    uint64_t n_bitmap_words;
    // record mode (stream_rec_kernel): one thread per record
    const uint64_t *offsets; // n_rec + 1
    uint64_t n_rec;
    uint32_t *counts;        // nullable: per-record hit counts
    uint32_t *fallback;      // device flag: record mode met a record above rec_limit -> the chunk kernels redo the batch
    uint32_t rec_limit;      // longest record one thread of stream_rec_kernel walks
    int chunk_blocks;        // chunk mode: 16-position blocks walked by one thread (2, 4 or 8: small batches use short chunks)
    // record mode, records above rec_limit: stream_rec_kernel lists them as groups of kLongGroup chunks of kLongChunk
    // positions, stream_long_kernel walks exactly those (the group counter is the word after `fallback`)
    uint2 *long_groups;      // nullable: (record, group index inside the record)
    uint32_t long_cap;       // entries long_groups holds; a batch that needs more falls back to the chunk kernels
};
constexpr uint32_t kLongChunk = 128; // positions per thread of stream_long_kernel, on the batch's 128-position grid
constexpr uint32_t kLongGroup = SBF_STREAM_TPB; // chunks per CTA

struct NaiveParams {
    StreamParams sp;
    int k, m, s, H;
};

__host__ __device__ constexpr uint64_t low_mask64(int nbits) { return nbits >= 64 ? ~0ull : ((1ull << nbits) - 1ull); }

template <int I, int N, class F>
__device__ __forceinline__ void static_for(F &&f)
{
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
}

// ---- the pinned primitives -----------------------------------------------------------------
// A1: minimizer order key of an m-mer ("lightweight multiplicative hash")
__device__ __forceinline__ uint32_t g_key(uint64_t x, int m)
{
    x ^= kSeedM & low_mask64(2 * m);
    return ((uint32_t)x ^ (uint32_t)(x >> 32)) * kMultG;
}
// A2: minimizer key -> shard (power-of-two shard count, no division)
__device__ __forceinline__ uint64_t sigma_shard(uint32_t key, int shard_shift)
{
    uint32_t t = (uint32_t)(((uint64_t)key * kGold64) >> 32);
    return (uint64_t)t >> shard_shift;
}
// A4: s-mer hash ("stronger mix with an additional xorshift")
__device__ __forceinline__ uint64_t f_hash(uint64_t x, int s)
{
    x ^= kSeedS & low_mask64(2 * s);
    uint64_t h = (x ^ (x >> 28)) * kMultF;
    return h ^ (h >> 32);
}
// the same value with the seed folded: ((x^sd) ^ ((x^sd)>>28)) = x ^ (x>>28) ^ (sd ^ (sd>>28))  (one LOP3 per half)
template <int S>
__device__ __forceinline__ uint64_t f_hash_c(uint64_t x)
{
    constexpr uint64_t sd = kSeedS & low_mask64(2 * S);
    constexpr uint64_t c = sd ^ (sd >> 28);
    uint64_t h = (x ^ (x >> 28) ^ c) * kMultF;
    return h ^ (h >> 32);
}
// A5 / A6: bit position of hash index i inside sector word i mod 4
__device__ __forceinline__ int bit_pos(uint64_t h, int i, int H)
{
    int W = 64 / H;
    if (W >= 6) return (int)((h >> (i * W)) & 63);
    return (int)((h * ((uint64_t)(2 * i + 1) * kGold64)) >> 58);
}

__device__ __forceinline__ void ld_shard_256(const uint64_t *p, uint64_t (&w)[4])
{
    // one 256-bit non-coherent load per shard: LDG.E.ENL2.256.CONSTANT on sm_100a
    asm volatile("ld.global.nc.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(w[0]), "=l"(w[1]), "=l"(w[2]), "=l"(w[3]) : "l"(p));
}

__device__ __forceinline__ void red_or_64(uint64_t *p, uint64_t v)
{
    asm volatile("red.global.or.b64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// One sector update as a single 32-byte TMA reduction (SASS UBLKRED): the four words go to a shared-memory slot of
// this thread and one cp.reduce.async.bulk ORs them into the filter.  Two slots per thread: before a slot is rewritten
// the bulk operation that read it two flushes ago must have finished reading (wait_group.read 1).
constexpr int kFlushSlots = 2;
__device__ __forceinline__ void tma_or_sector(uint64_t *dst, const uint64_t (&w)[4], ulonglong2 *slots, uint32_t &n_flushed)
{
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(kFlushSlots - 1) : "memory");
    ulonglong2 *s = slots + ((n_flushed & (kFlushSlots - 1)) * kStreamTPB + threadIdx.x) * 2; // [slot][thread][2 x 16 bytes]
    s[0] = make_ulonglong2(w[0], w[1]);
    s[1] = make_ulonglong2(w[2], w[3]);
    ++n_flushed;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    const uint32_t a0 = (uint32_t)__cvta_generic_to_shared(s);
    asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.or.b64 [%0], [%1], 32;" ::"l"(dst), "r"(a0) : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}

// =============================================================================================
// a1: pack.  Thread i produces packed words 2i, 2i+1 and the 32 V bits of symbols [32i, 32i+32).
//   code: A=0 C=1 G=2 T=3 (either case, A9); anything else is invalid (code bits arbitrary).
//   B[j] = symbol j is not ACGT, or j >= len.   V[j] = B[j] | B[j+1] | ... | B[j+k-1]:
//   no valid k-mer starts at symbol j.  Record ends are not known here: record mode bounds each
//   record by its own length, chunk mode over records adds them with mark_ends_kernel.
// =============================================================================================
__device__ __forceinline__ uint32_t pack4(uint32_t v, uint32_t &inv4)
{
    // four ASCII bytes (first symbol in the low byte) -> 8 bits, first symbol in the top 2 bits.
    // code = bits (b2, b1^b2) of the symbol: A 0, C 1, G 2, T 3 (either case).  Validity by the round trip: the
    // symbol is valid iff, with its case bit cleared, it EQUALS the letter of its own code — one byte permute
    // (PRMT as a 4-entry table "ACGT" indexed by the four codes) and one XOR instead of per-letter compares.
    // The gathers are byte dot products (IDP.4A), which run off the alu pipe this kernel is bound by.
    const uint32_t x = (v >> 1) & 0x03030303u;
    const uint32_t c = x ^ ((x >> 1) & 0x01010101u);
    const uint32_t sel = __dp4a(c, 0x00001001u, 0u) + (__dp4a(c, 0x10010000u, 0u) << 8); // the four codes as nibbles
    const uint32_t diff = (v & 0xDFDFDFDFu) ^ __byte_perm(0x54474341u, 0u, sel);
    // bit 7 of every byte of nz = that byte of diff is non-zero (no carry crosses a byte: 0x7F + 0x7F < 0x100)
    const uint32_t nz = (((diff & 0x7F7F7F7Fu) + 0x7F7F7F7Fu) | diff) & 0x80808080u;
    inv4 = __dp4a(nz, 0x08040201u, 0u) >> 7; // bit j = symbol j invalid
    return __dp4a(c, 0x01041040u, 0u);
}

// The same codes with the validity test deferred: returns TWICE the 8 code bits (bit 0 is zero) and ORs into `bad` the
// XOR of the four symbols (case bit cleared) with the letters of their own codes — zero iff all four are ACGT.  Almost
// every thread sees only valid symbols, so the per-symbol invalid flags (pack4) are only worked out when `bad` is not zero.
//   per byte t = 2 * code: bit 2 = b2, bit 1 = b1 ^ b2 (three instructions for four symbols); t indexes an 8-entry
//   byte table "A.C.G.T." directly (no shift), and the byte dot product gathers 2 * (c0 c1 c2 c3).
__device__ __forceinline__ uint32_t pack4_codes2(uint32_t v, uint32_t &bad)
{
    const uint32_t u = v & 0x06060606u;
    const uint32_t t = (u ^ (u >> 1)) & 0x06060606u;
    const uint32_t sel = __dp4a(t, 0x00001001u, 0u) + (__dp4a(t, 0x10010000u, 0u) << 8); // the four 2 * codes as nibbles
    uint32_t letters;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(letters) : "r"(0x00430041u), "r"(0x00540047u), "r"(sel));
    bad |= (v & 0xDFDFDFDFu) ^ letters;
    return __dp4a(t, 0x01041040u, 0u);
}

#ifdef SBF_DEFINE_AUX_KERNELS // non-template kernels: defined in one translation unit (sbf_api.cu)
// 32 symbols starting at b0 as eight little-endian 4-byte groups ('N' past the end)
__device__ __forceinline__ void load32(const uint8_t *__restrict__ seq, uint64_t b0, uint64_t len, int aligned16, uint32_t (&v)[8])
{
    if (aligned16 && b0 + 32 <= len) {
        const uint4 q0 = __ldg(reinterpret_cast<const uint4 *>(seq + b0));
        const uint4 q1 = __ldg(reinterpret_cast<const uint4 *>(seq + b0 + 16));
        v[0] = q0.x; v[1] = q0.y; v[2] = q0.z; v[3] = q0.w;
        v[4] = q1.x; v[5] = q1.y; v[6] = q1.z; v[7] = q1.w;
    } else {
#pragma unroll
        for (int w = 0; w < 8; ++w) {
            uint32_t acc = 0;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint64_t p = b0 + 4 * w + j;
                const uint32_t c = (p < len) ? (uint32_t)seq[p] : (uint32_t)'N';
                acc |= c << (8 * j);
            }
            v[w] = acc;
        }
    }
}

// bitmap_zero (nullable): the result bitmap of a record-mode query, whose word i covers exactly this thread's 32
// symbols — zeroed here, in passing, because record mode ORs into the words two records share.
// flag_zero (nullable): the record-mode fallback flag and, in the next word, the long-record group counter, cleared by
// the first thread.
__global__ void __launch_bounds__(256) pack_kernel(const uint8_t *__restrict__ seq, uint64_t len, uint32_t *__restrict__ packed,
                                                   uint16_t *__restrict__ vmask, uint64_t n_words_total, int k, int aligned16,
                                                   uint32_t *__restrict__ bitmap_zero, uint64_t n_bitmap_words,
                                                   uint32_t *__restrict__ flag_zero)
{
    // thread i: symbols [32i, 32i+32) -> packed words 2i, 2i+1 (one 8-byte store) and their two mask words (one 4-byte store)
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t b0 = i * 32;
    if (i == 0 && flag_zero != nullptr) { flag_zero[0] = 0; flag_zero[1] = 0; } // fallback flag, long-record group counter
    uint32_t v[8];
    load32(seq, b0, len, aligned16, v);
    uint32_t word[2] = {0, 0}, inv = 0, bad = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
        const uint32_t c9 = pack4_codes2(v[w], bad); // 2 * (8 code bits)
        word[w >> 2] |= (w & 3) == 3 ? c9 >> 1 : c9 << (23 - 8 * (w & 3));
    }
    if (bad != 0) { // some symbol of these 32 is not ACGT (or lies past the end): which ones
#pragma unroll
        for (int w = 0; w < 8; ++w) {
            uint32_t i4;
            (void)pack4(v[w], i4);
            inv |= i4 << (4 * w);
        }
    }
    // B of the next 32 (k > 33: 64) symbols: the following threads' words through shared memory; only the last thread(s)
    // of the CTA classify them themselves (a per-warp exchange would send one lane in 32 down that divergent path)
    __shared__ uint32_t s_inv[256];
    s_inv[threadIdx.x] = inv;
    __syncthreads();
    auto inv_ahead = [&](unsigned d) -> uint32_t { // B bits of symbols [b0 + 32 d, b0 + 32 d + 32)
        if (threadIdx.x + d < blockDim.x) return s_inv[threadIdx.x + d];
        uint32_t vv[8], r = 0;
        load32(seq, b0 + 32ull * d, len, aligned16, vv);
#pragma unroll
        for (int w = 0; w < 8; ++w) {
            uint32_t i4;
            (void)pack4(vv[w], i4);
            r |= i4 << (4 * w);
        }
        return r;
    };
    const uint32_t nxt = inv_ahead(1);
    // V = OR of k consecutive B bits, by doubling: after the loop bit j of y covers B[j .. j+c-1], c the largest power
    // of two <= k; one more step with the remainder closes the window (k - c <= c)
    uint32_t g;
    if (k <= 33) {
        uint64_t y = (uint64_t)inv | ((uint64_t)nxt << 32);
        if (__any_sync(0xFFFFFFFFu, y != 0)) { // almost every warp sees only valid symbols: V = 0 without the doubling
            int c = 1;
            while (2 * c <= k) {
                y |= y >> c;
                c *= 2;
            }
            if (c < k) y |= y >> (k - c);
        }
        g = (uint32_t)y;
    } else { // 33 < k <= 64: the window reaches into the third word
        unsigned __int128 y = (unsigned __int128)inv | ((unsigned __int128)nxt << 32) | ((unsigned __int128)inv_ahead(2) << 64);
        int c = 1;
        while (2 * c <= k) {
            y |= y >> c;
            c *= 2;
        }
        if (c < k) y |= y >> (k - c);
        g = (uint32_t)y;
    }
    if (2 * i + 1 < n_words_total) {
        *reinterpret_cast<uint2 *>(packed + 2 * i) = make_uint2(word[0], word[1]);
        *reinterpret_cast<uint32_t *>(vmask + 2 * i) = g;
    } else if (2 * i < n_words_total) {
        packed[2 * i] = word[0];
        vmask[2 * i] = (uint16_t)g;
    }
    if (bitmap_zero != nullptr && i < n_bitmap_words) bitmap_zero[i] = 0;
}

// Chunk mode over a record batch: the k-1 start positions before a record end e = offsets[r] (r = 1..n_rec) have no
// k-mer (it would span two records): OR the bit range [e-(k-1), e) into V.  only_if (nullable): the record-mode
// fallback flag — the launch does nothing unless it is set.
__global__ void __launch_bounds__(256) mark_ends_kernel(const uint64_t *__restrict__ offsets, uint64_t n_rec, uint64_t total,
                                                        uint32_t *vmask32, int k, const uint32_t *only_if)
{
    if (only_if != nullptr && *only_if == 0) return;
    for (uint64_t r = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x + 1; r <= n_rec; r += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t e = offsets[r];
        if (k < 2 || e == 0 || e > total) continue;
        const uint64_t lo = e >= (uint64_t)(k - 1) ? e - (uint64_t)(k - 1) : 0;
        // at most k - 1 <= 63 bits starting at bit (lo & 31): at most three words
        const unsigned __int128 mask = ((((unsigned __int128)1) << (e - lo)) - 1) << (lo & 31);
        atomicOr(&vmask32[lo >> 5], (uint32_t)mask);
        if ((uint32_t)(mask >> 32)) atomicOr(&vmask32[(lo >> 5) + 1], (uint32_t)(mask >> 32));
        if ((uint32_t)(mask >> 64)) atomicOr(&vmask32[(lo >> 5) + 2], (uint32_t)(mask >> 64));
    }
}

#endif // SBF_DEFINE_AUX_KERNELS

// =============================================================================================
// Window access for stream_kernel.  W[0..NWIN-1] hold 16 * NWIN consecutive symbols (W[0] first, first symbol in the
// top bits).  lmer<O,N>(W) = the N-mer starting O symbols into the window, as Sub() of the paper's packed k-mer (first
// base most significant); an N-mer wider than 64 bits (N > 32: k-mers of 33..64 bases, A20) comes back folded to
// 64 bits as A21 prescribes (its last 32 symbols XOR the rotated golden-ratio multiple of the symbols before them).
// All shifts are immediates.  NWIN = 4 up to k = 42, 5 up to k = 58, 6 up to k = 64 (kWinOf).
// =============================================================================================
__host__ __device__ constexpr int kWinOf(int K) { return (K + 15 + SBF_Q_LA + 15) / 16 < 4 ? 4 : (K + 15 + SBF_Q_LA + 15) / 16; } // 15 + look-ahead + k symbols

template <int Q, int NB, int NWIN>
__device__ __forceinline__ uint32_t field_win(const uint32_t (&W)[NWIN])
{
    // bits [Q, Q+NB) of the window, counted from the least significant bit of W[NWIN-1]
    static_assert(Q >= 0 && NB >= 1 && NB <= 32 && Q + NB <= 32 * NWIN, "field outside the register window");
    constexpr int idx = Q / 32, sh = Q % 32;
    uint32_t lo = W[NWIN - 1 - idx];
    uint32_t v;
    if constexpr (sh == 0) {
        v = lo;
    } else if constexpr (sh + NB <= 32) {
        v = lo >> sh;
    } else {
        v = __funnelshift_r(lo, W[NWIN - 2 - idx], sh);
    }
    if constexpr (NB < 32 && !(sh + NB == 32)) v &= (1u << NB) - 1u;
    return v;
}

template <int O, int N, int NWIN>
__device__ __forceinline__ uint64_t lmer(const uint32_t (&W)[NWIN])
{
    if constexpr (N <= 32) {
        constexpr int Q = 32 * NWIN - 2 * O - 2 * N;
        constexpr int nb = 2 * N;
        uint32_t lo = field_win<Q, (nb < 32 ? nb : 32)>(W);
        uint32_t hi = 0;
        if constexpr (nb > 32) hi = field_win<Q + 32, nb - 32>(W);
        return ((uint64_t)hi << 32) | lo;
    } else {
        const uint64_t lo = lmer<O + (N - 32), 32>(W); // the last 32 symbols: the low 64 bits of the window
        const uint64_t hi = lmer<O, N - 32>(W);        // the symbols before them: the bits above
        const uint64_t t = hi * kGold64;
        return lo ^ ((t << 32) | (t >> 32));
    }
}

// three-input minimum as an opaque pair of min.u32 (ptxas fuses it into one VIMNMX3); written with min(min(a, b), c)
// the optimiser re-associates the sliding-minimum tree across positions into two-input minima — about twice as many
__device__ __forceinline__ uint32_t min3u(uint32_t a, uint32_t b, uint32_t c)
{
#if SBF_MIN3_ASM
    uint32_t r;
    asm("{\n\t.reg .u32 t;\n\tmin.u32 t, %1, %2;\n\tmin.u32 %0, t, %3;\n\t}" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
#else
    return min(min(a, b), c);
#endif
}

// Sliding minimum of the last WN keys, streaming: keys arrive one per step, E = step phase (mod 16
// is all that matters).  Levels c3 = min of the last 3, c9 = min of the last 9; the window of WN is
// covered by two or three overlapping blocks (three-input minimum = VIMNMX3 on sm_100a); above 24 keys (k-mers of more
// than 32 bases with m near k/2) a fourth level keeps the minimum of the last 24 and joins it with an earlier one.
template <int WN>
struct SlidingMin {
    static_assert(WN >= 1 && WN <= 39, "stream kernel supports k-m+1 <= 39");
    uint32_t g[16], c3[16], c9[16], c24[16];
    __device__ __forceinline__ void clear()
    {
#pragma unroll
        for (int i = 0; i < 16; ++i) { g[i] = 0; c3[i] = 0; c9[i] = 0; c24[i] = 0; }
    }
    template <int E>
    __device__ __forceinline__ uint32_t push(uint32_t gn)
    {
        constexpr int s0 = E & 15;
        g[s0] = gn;
        if constexpr (WN == 1) return gn;
        if constexpr (WN == 2) return min(gn, g[(E - 1) & 15]);
        uint32_t a3 = min3u(gn, g[(E - 1) & 15], g[(E - 2) & 15]);
        c3[s0] = a3;
        if constexpr (WN == 3) return a3;
        if constexpr (WN >= 4 && WN <= 6) return min(a3, c3[(E - (WN - 3)) & 15]);
        if constexpr (WN >= 7 && WN <= 9) return min3u(a3, c3[(E - 3) & 15], c3[(E - (WN - 3)) & 15]);
        if constexpr (WN >= 10) {
            uint32_t a9 = min3u(a3, c3[(E - 3) & 15], c3[(E - 6) & 15]);
            c9[s0] = a9;
            if constexpr (WN <= 18) return min(a9, c9[(E - (WN - 9)) & 15]);
            else if constexpr (WN <= 24) return min3u(a9, c9[(E - 9) & 15], c9[(E - (WN - 9)) & 15]);
            else {
                const uint32_t a24 = min3u(a9, c9[(E - 9) & 15], c9[(E - 15) & 15]);
                c24[s0] = a24;
                return min(a24, c24[(E - (WN - 24)) & 15]);
            }
        }
        return gn;
    }
};

// Sliding OR of the last WO masks (WO = k-s+1: the k-mer's mask K is the OR of its s-mers' one-hot masks), streaming like
// SlidingMin: c3 = OR of the last 3, c9 = OR of the last 9, the window covered by two or three overlapping blocks —
// overlap is free for OR, and a three-input OR (or OR-then-AND-NOT) is one LOP3.  push_test() returns the bits of K
// that are NOT set in the shard (all zero = every s-mer of the k-mer hits, the Findere rule).
template <int WO, int NW>
struct SlidingOr {
    static_assert(WO >= 1 && WO <= 17, "stream kernels support k-s <= 16");
    uint64_t m[16][NW], c3[16][NW], c9[16][NW];
    __device__ __forceinline__ void clear()
    {
#pragma unroll
        for (int i = 0; i < 16; ++i)
#pragma unroll
            for (int q = 0; q < NW; ++q) { m[i][q] = 0; c3[i][q] = 0; c9[i][q] = 0; }
    }
    template <int E>
    __device__ __forceinline__ uint64_t window(const uint64_t (&Mn)[NW], int q)
    {
        constexpr int e = E & 15;
        m[e][q] = Mn[q];
        if constexpr (WO == 1) return Mn[q];
        if constexpr (WO == 2) return Mn[q] | m[(E - 1) & 15][q];
        const uint64_t a3 = Mn[q] | m[(E - 1) & 15][q] | m[(E - 2) & 15][q];
        c3[e][q] = a3;
        if constexpr (WO == 3) return a3;
        if constexpr (WO >= 4 && WO <= 6) return a3 | c3[(E - (WO - 3)) & 15][q];
        if constexpr (WO >= 7 && WO <= 9) return a3 | c3[(E - 3) & 15][q] | c3[(E - (WO - 3)) & 15][q];
        if constexpr (WO >= 10) {
            const uint64_t a9 = a3 | c3[(E - 3) & 15][q] | c3[(E - 6) & 15][q];
            c9[e][q] = a9;
            return a9 | c9[(E - (WO - 9)) & 15][q];
        }
        return a3;
    }
    template <int E>
    __device__ __forceinline__ void push(const uint64_t (&Mn)[NW])
    {
#pragma unroll
        for (int q = 0; q < NW; ++q) (void)window<E>(Mn, q);
    }
    template <int E>
    __device__ __forceinline__ uint64_t push_test(const uint64_t (&Mn)[NW], const uint64_t (&shard)[4])
    {
        uint64_t miss = 0;
#pragma unroll
        for (int q = 0; q < NW; ++q) miss |= window<E>(Mn, q) & ~shard[q];
        return miss;
    }
};

// Sliding Findere test WITHOUT 256-bit masks (query, H <= 4, k-s+1 in {1, 2, 4, 8}).  A bit position B(h,i) of sector
// word q = i is (byte y = B >> 3, bit z = B & 7).  Per word q the thread keeps, for the last WO s-mers (ring slot
// r = s-mer index mod WO, four slots per register):
//   S[q] : four selector nibbles, nibble r = y of slot r   -> ONE byte permute G = PRMT(word q lo, word q hi, S[q])
//          gathers, from the CURRENT shard, the byte each of the four s-mers must hit in word q;
//   T[q] : four bytes, byte r = 1 << z of slot r           -> T[q] & ~G = bits of word q the k-mer misses.
// Nothing here depends on the shard, so a shard change costs nothing (the gather always reads the current shard
// registers), exactly like the mask form — but the state is 2 registers per word instead of ~6, and a position costs
// ~21 alu-pipe instructions instead of ~37 (8 variable 64-bit shifts for the one-hot masks and 24 LOP3 for the sliding
// OR and the AND-NOT over eight 32-bit halves are gone).  New s-mer, slot r: the y fields go into nibble r of S[q]
// with one shift and one masked insert (LOP3) per word; the four z fields are packed into selector nibbles
// (PRMT + mask + one multiply-add-high on the fma pipe), one table PRMT turns them into four one-hot bytes, and one
// PRMT per word puts byte q of that into byte r of T[q].
// prmt.b32 as is (__byte_perm would first AND the selector with 0x7777: one more LOP3 per use); selector nibbles must be 0..7
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel)
{
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
    return d;
}
// (a & mask) | (b & ~mask) as ONE LOP3 (written out, the compiler spends two: it sees two different constants)
__device__ __forceinline__ uint32_t bitsel(uint32_t a, uint32_t b, uint32_t mask)
{
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0xE4;" : "=r"(d) : "r"(a), "r"(b), "r"(mask));
    return d;
}

template <int WO, int H>
struct SlidingGather {
    static_assert(H >= 1 && H <= 4 && (WO == 1 || WO == 2 || WO == 4 || WO == 8), "gather form: H <= 4, k-s+1 in {1,2,4,8}");
    static constexpr int NW = H, Wd = 64 / H, NSET = WO > 4 ? 2 : 1;
    static constexpr bool PAIRED = SBF_GATHER_PAIRED != 0 && H == 4;
    uint32_t S[NSET][NW], T[NSET][NW];
    __device__ __forceinline__ void clear()
    {
#pragma unroll
        for (int a = 0; a < NSET; ++a)
#pragma unroll
            for (int q = 0; q < NW; ++q) { S[a][q] = 0; T[a][q] = 0; }
    }
    template <int SH>
    __device__ __forceinline__ static uint32_t shift_to(uint32_t x) // x >> SH (SH > 0) or x << -SH
    {
        if constexpr (SH == 0) return x;
        else if constexpr (SH > 0) {
#if SBF_GATHER_FMA_SHIFT
            return __umulhi(x, 1u << (32 - SH));
#else
            return x >> SH;
#endif
        } else return x << (-SH);
    }
    // the four (H) z fields of hash h as clean selector nibbles, nibble q = z of word q
    __device__ __forceinline__ static uint32_t z_nibbles(uint32_t lo, uint32_t hi)
    {
        if constexpr (H == 4) { // fields at bits 0, 16 (lo), 0, 16 (hi): bytes (lo.b0, hi.b0, lo.b2, hi.b2), then byte 2 -> nibble 1, byte 1 -> nibble 2
            const uint32_t pm = prmt(lo, hi, 0x6240u) & 0x07070707u;
            uint32_t zs;
            asm("mad.hi.u32 %0, %1, %2, %1;" : "=r"(zs) : "r"(pm), "r"(1u << 20)); // pm | (pm >> 12); bits above 15 are ignored by PRMT
            return zs;
        } else if constexpr (H == 2) { // fields at bit 0 of lo and of hi
            return (lo & 7u) | ((hi & 7u) << 4);
        } else if constexpr (H == 1) {
            return lo & 7u;
        } else {
            uint32_t zs = 0;
            static_for<0, H>([&](auto qc) {
                constexpr int q = decltype(qc)::value, off = q * Wd;
                zs |= (((off < 32 ? lo : hi) >> (off % 32)) & 7u) << (4 * q);
            });
            return zs;
        }
    }
    template <int E>
    __device__ __forceinline__ void push(uint64_t h)
    {
        constexpr int r = E % WO, a = r / 4, rr = r % 4;
        const uint32_t lo = (uint32_t)h, hi = (uint32_t)(h >> 32);
        const uint32_t onehot = prmt(0x08040201u, 0x80402010u, z_nibbles(lo, hi)); // byte q = 1 << z of word q
        static_for<0, NW>([&](auto qc) {
            constexpr int q = decltype(qc)::value, off = q * Wd;
            static_assert(off % 32 + 6 <= 32, "a 6-bit slice straddles the halves of the hash");
            if constexpr (PAIRED) {
                // H = 4: the fields of words q and q+1 sit 16 bits apart in one half of the hash, so ONE shift and ONE
                // masked insert serve both: S[q] keeps word q's selector in its low half and word q+1's in its high half
                if constexpr ((q & 1) == 0) {
                    constexpr uint32_t nib2 = 0x00070007u << (4 * rr);
                    S[a][q] = bitsel(shift_to<3 - 4 * rr>(q < 2 ? lo : hi), S[a][q], nib2);
                }
            } else {
                constexpr uint32_t nib = 7u << (4 * rr);
                const uint32_t y = shift_to<off % 32 + 3 - 4 * rr>(off < 32 ? lo : hi); // y field moved to nibble rr, junk around it
                S[a][q] = bitsel(y, S[a][q], nib);
            }
            constexpr uint32_t keep = 0x3210u & ~(0xFu << (4 * rr)); // T[q] bytes stay, byte rr <- onehot byte q
            T[a][q] = prmt(T[a][q], onehot, keep | ((uint32_t)(4 + q) << (4 * rr)));
        });
    }
    __device__ __forceinline__ uint32_t selector(int a, int q) const
    {
        if constexpr (PAIRED) {
            if (q & 1) {
#if SBF_GATHER_FMA_SHIFT
                return __umulhi(S[a][q - 1], 1u << 16);
#else
                return S[a][q - 1] >> 16;
#endif
            }
        }
        return S[a][q];
    }
    // bits of the k-mer's H * WO positions that are NOT set in the shard (0 = present); sh32 = the sector as 8 halves
    template <int E>
    __device__ __forceinline__ uint32_t push_test(uint64_t h, const uint32_t (&sh32)[8])
    {
        push<E>(h);
        uint32_t miss = 0;
#pragma unroll
        for (int a = 0; a < NSET; ++a)
#pragma unroll
            for (int q = 0; q < NW; ++q) miss |= T[a][q] & ~prmt(sh32[2 * q], sh32[2 * q + 1], selector(a, q));
        return miss;
    }
};
template <int WO, int H>
constexpr bool gather_form() { return SBF_GATHER != 0 && H <= 4 && (WO == 1 || WO == 2 || WO == 4 || WO == 8); }

// 1 << b for b in [0, 64) as two 32-bit halves.  SBF_FMA_ONEHOT: one shift on the alu pipe (1 << (b & 31)), the
// half it belongs to picked by multiplications (b >> 5 as a multiply-high, then x * {0,1} and x - y as IMADs), which
// issue on the fma pipe — the stream kernels are bound by the alu pipe, the fma pipe is two thirds idle.
__device__ __forceinline__ uint64_t onehot64(uint32_t b)
{
#if SBF_FMA_ONEHOT
    const uint32_t m32 = 1u << (b & 31u);
    const uint32_t b5 = __umulhi(b, 0x08000000u); // b >> 5
    uint32_t hi, lo;
    asm("mul.lo.u32 %0, %1, %2;" : "=r"(hi) : "r"(m32), "r"(b5));
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(lo) : "r"(hi), "r"(0xFFFFFFFFu), "r"(m32)); // m32 - hi
    return ((uint64_t)hi << 32) | lo;
#else
    return 1ull << b;
#endif
}

// One-hot sector masks of one s-mer hash: hash index i -> word i mod 4, bit B(h,i) (A5)
template <int OFF>
__device__ __forceinline__ uint64_t onehot_at(uint64_t h)
{
#if SBF_IDP_EXTRACT
    if constexpr (OFF % 8 == 0) {
        // byte-aligned slice: mask all four bytes of the half at once (shared by the other slices of that half), then
        // pick the byte with a byte dot product (IDP.4A runs off the alu pipe that bounds the query kernels)
        const uint32_t half = OFF < 32 ? (uint32_t)h : (uint32_t)(h >> 32);
        return onehot64(__dp4a(half & 0x3F3F3F3Fu, 1u << (OFF % 32), 0u));
    }
#endif
    return onehot64((uint32_t)(h >> OFF) & 63u);
}

template <int H, int NW>
__device__ __forceinline__ void expand_masks(uint64_t h, uint64_t (&m)[NW])
{
    constexpr int Wd = 64 / H;
    static_assert(Wd >= 6, "bit-slicing needs 64/H >= 6");
#pragma unroll
    for (int q = 0; q < NW; ++q) m[q] = 0;
    static_for<0, H>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        m[i & 3] |= onehot_at<i * Wd>(h);
    });
}

__host__ __device__ constexpr int ring_size(int z) { return z <= 1 ? 1 : z <= 2 ? 2 : z <= 4 ? 4 : z <= 8 ? 8 : 16; }

// A2.  shard_shift = 32 - P (32 when there is one shard).  The final shift t >> (32 - P) is a multiply-high by 2^P
// on the fma pipe (specialised kernels serve P <= 31; 2^32 shards run the runtime-parameter kernel).
__device__ __forceinline__ uint32_t sigma32(uint32_t key, int shard_shift)
{
    uint32_t t = (uint32_t)(((uint64_t)key * kGold64) >> 32);
#if SBF_FMA_SIGMA
    return __umulhi(t, 1u << ((32 - shard_shift) & 31));
#else
    return __funnelshift_rc(t, 0u, (uint32_t)shard_shift);
#endif
}

// query staging through shared memory: the 32 bytes of a shard travel global -> shared with two 16-byte cp.async
// (LDGSTS, no register in between) kLA positions before the run's first test reads them back.
constexpr int kLA = SBF_Q_LA; // the minimizer runs this many positions ahead of the bit tests
constexpr int kNS = kLA + 1;  // staging slots per thread: k-mer q uses slot q mod kNS
static_assert(kLA >= 1 && 16 % kNS == 0, "staging needs a look-ahead of 1, 3, 7 or 15");

__device__ __forceinline__ void cp_async_shard(uint4 *smem_lo, uint4 *smem_hi, const uint64_t *g)
{
    uint32_t a = (uint32_t)__cvta_generic_to_shared(smem_lo), b = (uint32_t)__cvta_generic_to_shared(smem_hi);
#if SBF_CPASYNC_L2_64B
    asm volatile("cp.async.cg.shared.global.L2::64B [%0], [%1], 16;" ::"r"(a), "l"(g) : "memory");
    asm volatile("cp.async.cg.shared.global.L2::64B [%0], [%1], 16;" ::"r"(b), "l"(g + 2) : "memory");
#else
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(a), "l"(g) : "memory");
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(b), "l"(g + 2) : "memory");
#endif
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// The query pipeline of one thread (shared by chunk mode and record mode): minimizer + shard of k-mer q+kLA, staging
// of a new run's sector, the newest s-mer's masks, the k-mer test of k-mer q.  Validity plays no part here: a
// position without a valid k-mer computes on whatever symbols are there (its shard index is still in range) and its
// result bit is cleared from V afterwards, 16 positions at a time.
template <int K, int M, int S, int H, int TPB>
struct QueryLane {
    static constexpr int WN = K - M + 1, Z = K - S, NW = H < 4 ? H : 4, NWIN = kWinOf(K);
    static constexpr bool GATHER = gather_form<Z + 1, H>();
    SlidingMin<WN> smin;
    std::conditional_t<GATHER, SlidingGather<GATHER ? Z + 1 : 1, GATHER ? H : 1>, SlidingOr<Z + 1, NW>> sor;
    uint32_t sh32[8]; // the current shard's four sector words as 32-bit halves (little-endian)
    uint32_t laPrev;
    bool sb[kNS]; // sb[q mod kNS]: a run starts at k-mer q (its sector is in staging slot q mod kNS)

    // keys of the first WN-1 m-mers, masks of the first Z s-mers, shards of the first kLA k-mers
    __device__ __forceinline__ void prologue(const uint32_t (&W)[NWIN], const StreamParams &prm, uint4 *stage)
    {
        smin.clear();
        sor.clear();
#pragma unroll
        for (int q = 0; q < 8; ++q) sh32[q] = 0;
#pragma unroll
        for (int i = 0; i < kNS; ++i) sb[i] = false;
        laPrev = 0;
        static_for<0, WN - 1>([&](auto ec) {
            constexpr int E = decltype(ec)::value;
            (void)smin.template push<E>(g_key(lmer<E, M>(W), M));
        });
        static_for<0, Z>([&](auto ic) {
            constexpr int I = decltype(ic)::value;
            if constexpr (GATHER) {
                sor.template push<I>(f_hash_c<S>(lmer<I, S>(W)));
            } else {
                uint64_t Mi[NW];
                expand_masks<H, NW>(f_hash_c<S>(lmer<I, S>(W)), Mi);
                sor.template push<I>(Mi);
            }
        });
        static_for<0, kLA>([&](auto qc) { this->template look<decltype(qc)::value, decltype(qc)::value == 0>(W, prm, stage); });
    }
    // k-mer Q (relative to the window): its shard; a change of shard starts a run and stages that sector
    template <int Q, bool FIRST>
    __device__ __forceinline__ void look(const uint32_t (&W)[NWIN], const StreamParams &prm, uint4 *stage)
    {
        const uint32_t shNew = sigma32(smin.template push<Q + WN - 1>(g_key(lmer<Q + WN - 1, M>(W), M)), prm.shard_shift);
        const bool start = FIRST || shNew != laPrev;
        if (start)
            cp_async_shard(&stage[((Q % kNS) * 2) * TPB + threadIdx.x], &stage[((Q % kNS) * 2 + 1) * TPB + threadIdx.x],
                           prm.filter + (uint64_t)shNew * 4);
        cp_async_commit();
        sb[Q % kNS] = start;
        laPrev = shNew;
    }
    // k-mer J of the current 16-position block: returns 0 iff all its H(k-s+1) bits are set in its shard
    template <int J>
    __device__ __forceinline__ uint32_t step(const uint32_t (&W)[NWIN], const StreamParams &prm, uint4 *stage)
    {
        // a6: if a run starts here, its sector was staged kLA positions ago: take it into the shard registers.
#if SBF_PRED_RELOAD
        // Almost every warp has SOME lane starting a run at any given position, so a branch would be taken (and its
        // BSSY/BSYNC paid) nearly always: wait unconditionally, load under a predicate.  SBF_EARLY_RELOAD: do it FIRST
        // in the step (before this step's own look-ahead commits its group, hence wait_group kLA - 1), so that the
        // shared-memory latency hides behind the minimizer and hash work instead of in front of the test.
#if SBF_EARLY_RELOAD
        cp_async_wait<kLA - 1>();
#else
        this->template look<J + kLA, false>(W, prm, stage);
        cp_async_wait<kLA>();
#endif
        {
            const uint32_t a0 = (uint32_t)__cvta_generic_to_shared(&stage[((J % kNS) * 2) * TPB + threadIdx.x]);
            const uint32_t a1 = (uint32_t)__cvta_generic_to_shared(&stage[((J % kNS) * 2 + 1) * TPB + threadIdx.x]);
            asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %8, 0;\n\t"
                         "@p ld.shared.v4.u32 {%0,%1,%2,%3}, [%9];\n\t@p ld.shared.v4.u32 {%4,%5,%6,%7}, [%10];\n\t}"
                         : "+r"(sh32[0]), "+r"(sh32[1]), "+r"(sh32[2]), "+r"(sh32[3]), "+r"(sh32[4]), "+r"(sh32[5]), "+r"(sh32[6]),
                           "+r"(sh32[7])
                         : "r"((uint32_t)sb[J % kNS]), "r"(a0), "r"(a1)
                         : "memory");
        }
#if SBF_EARLY_RELOAD
        this->template look<J + kLA, false>(W, prm, stage);
#endif
#else
        this->template look<J + kLA, false>(W, prm, stage);
        if (sb[J % kNS]) {
            cp_async_wait<kLA>();
            const uint4 lo = stage[((J % kNS) * 2) * TPB + threadIdx.x];
            const uint4 hi = stage[((J % kNS) * 2 + 1) * TPB + threadIdx.x];
            sh32[0] = lo.x; sh32[1] = lo.y; sh32[2] = lo.z; sh32[3] = lo.w;
            sh32[4] = hi.x; sh32[5] = hi.y; sh32[6] = hi.z; sh32[7] = hi.w;
        }
#endif
        if constexpr (GATHER) {
            return sor.template push_test<J + Z>(f_hash_c<S>(lmer<J + Z, S>(W)), sh32);
        } else {
            uint64_t Mn[NW];
            expand_masks<H, NW>(f_hash_c<S>(lmer<J + Z, S>(W)), Mn);
            const uint64_t shard[4] = {((uint64_t)sh32[1] << 32) | sh32[0], ((uint64_t)sh32[3] << 32) | sh32[2],
                                       ((uint64_t)sh32[5] << 32) | sh32[4], ((uint64_t)sh32[7] << 32) | sh32[6]};
            const uint64_t miss = sor.template push_test<J + Z>(Mn, shard);
            return (uint32_t)miss | (uint32_t)(miss >> 32);
        }
    }
};

// =============================================================================================
// a2-a6 fused, CHUNK MODE.  One thread walks 16 * chunk_blocks consecutive k-mer start positions of the
// batch, carrying in registers: the 64-symbol window, the sliding-minimum rings (a2), the one-hot
// masks of the last k-s s-mers, and
//   insert: the OR of the current super-k-mer's masks (a5), flushed with one RED.OR.B64 per sector
//           word when the shard (A14) or validity changes;
//   query : the current shard's 256 bits (a6) and the sliding OR of the k-mer mask K, tested with
//           K & ~shard == 0 (Findere rule); see QueryLane.
// Each m-mer key and each s-mer hash is computed once per position (not once per k-mer as in
// Alg. 1/2); the result bits are the same because OR/AND do not care about order or repetition.
// =============================================================================================
// MODE: kModeQuery, kModeInsert (flush = four RED.OR.B64), kModeInsertTma (flush = one 32-byte TMA reduction: faster
// once the filter is much larger than L2 — the LSU path then spends four L2 requests on a sector that one DRAM
// read-modify-write serves; slower while the filter is L2-resident, where the TMA unit's ~24 G operations/s cap binds).
constexpr int kModeQuery = 0, kModeInsert = 1, kModeInsertTma = 2;
template <int K, int M, int S, int H, int MODE>
__global__ void __launch_bounds__(kStreamTPB, MODE != kModeQuery ? SBF_MINB_I : (gather_form<K - S + 1, H>() && K <= 32 ? SBF_MINB_Q : 4))
    stream_kernel(const StreamParams prm)
{
    constexpr bool INSERT = MODE != kModeQuery;
    constexpr bool TMA_FLUSH = MODE == kModeInsertTma;
    constexpr int WN = K - M + 1;
    constexpr int Z = K - S;
    constexpr int NW = H < 4 ? H : 4;
    constexpr int RZ = ring_size(Z);
    constexpr int NWIN = kWinOf(K);
    static_assert(K >= 1 && K <= 64 && M >= 1 && M <= K && S >= 1 && S <= K, "bad k/m/s");
    static_assert(Z <= 16, "stream kernel supports k-s <= 16");
    __shared__ uint4 stage[INSERT ? 1 : kNS * 2 * kStreamTPB];
    __shared__ ulonglong2 flush_slots[TMA_FLUSH ? kFlushSlots * kStreamTPB * 2 : 1];
    uint32_t n_flushed = 0;
    (void)flush_slots; (void)n_flushed;

    if constexpr (!INSERT) {
        if (prm.fallback != nullptr && *prm.fallback == 0) return; // stream_rec_kernel did this batch
    }
    // one chunk per thread; the (normally idle) fallback launch behind record mode uses a small grid and strides
    for (uint64_t chunk = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;; chunk += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t p0 = chunk * (uint64_t)(16 * prm.chunk_blocks);
    if (p0 >= prm.n_pos) return;

    const uint32_t *__restrict__ pw = prm.packed + (p0 >> 4);
    const uint16_t *__restrict__ vw = prm.vmask + (p0 >> 4);
    uint32_t W[NWIN];
#pragma unroll
    for (int i = 0; i < NWIN; ++i) W[i] = __ldg(pw + i);

    if constexpr (INSERT) {
        SlidingMin<WN> smin;
        smin.clear();
        uint64_t Mh[RZ][NW]; // masks of the last k-s s-mers: what a new run shares with the k-mers before it
#pragma unroll
        for (int i = 0; i < RZ; ++i)
#pragma unroll
            for (int q = 0; q < NW; ++q) Mh[i][q] = 0;
        static_for<0, WN - 1>([&](auto ec) {
            constexpr int E = decltype(ec)::value;
            (void)smin.template push<E>(g_key(lmer<E, M>(W), M));
        });
        static_for<0, Z>([&](auto ic) {
            constexpr int I = decltype(ic)::value;
            expand_masks<H, NW>(f_hash_c<S>(lmer<I, S>(W)), Mh[I % RZ]);
        });
        uint64_t acc[NW]; // OR of the current run's masks
#pragma unroll
        for (int q = 0; q < NW; ++q) acc[q] = 0;
        uint32_t prevShard = 0;
        bool prevInval = true;
        for (int b = 0; b < prm.chunk_blocks; ++b) {
            const uint32_t wnext = __ldg(pw + b + NWIN);
            const uint32_t v16 = __ldg(vw + b);
            static_for<0, 16>([&](auto jc) {
                constexpr int J = decltype(jc)::value;
                // a2/a3: key of the newest m-mer of k-mer p = p0+16b+J, its window minimum, its shard
                const uint32_t sh = sigma32(smin.template push<J + WN - 1>(g_key(lmer<J + WN - 1, M>(W), M)), prm.shard_shift);
                // a4: the newest s-mer of k-mer p
                uint64_t Mn[NW];
                expand_masks<H, NW>(f_hash_c<S>(lmer<J + Z, S>(W)), Mn);
                // a1: validity of k-mer p
                const bool inval = (v16 & (1u << J)) != 0;
                const bool brk = (sh != prevShard) || (inval != prevInval);
                if (brk) {
                    if (!prevInval) { // a5: flush the finished run
                        uint64_t *dst = prm.filter + (uint64_t)prevShard * 4;
                        if constexpr (TMA_FLUSH) {
                            const uint64_t w4[4] = {acc[0], NW > 1 ? acc[NW > 1 ? 1 : 0] : 0, NW > 2 ? acc[NW > 2 ? 2 : 0] : 0,
                                                    NW > 3 ? acc[NW > 3 ? 3 : 0] : 0};
                            tma_or_sector(dst, w4, flush_slots, n_flushed);
                        } else {
#pragma unroll
                            for (int q = 0; q < NW; ++q) red_or_64(dst + q, acc[q]);
                        }
                    }
#pragma unroll
                    for (int q = 0; q < NW; ++q) { // restart with the k-s s-mers shared with the previous k-mers
                        uint64_t r = 0;
#pragma unroll
                        for (int i = 0; i < Z; ++i) r |= Mh[(J + i) % RZ][q];
                        acc[q] = r;
                    }
                }
#pragma unroll
                for (int q = 0; q < NW; ++q) acc[q] |= Mn[q];
                prevShard = sh;
                prevInval = inval;
#pragma unroll
                for (int q = 0; q < NW; ++q) Mh[(J + Z) % RZ][q] = Mn[q];
            });
#pragma unroll
            for (int i = 0; i + 1 < NWIN; ++i) W[i] = W[i + 1];
            W[NWIN - 1] = wnext;
        }
        if (!prevInval) {
            uint64_t *dst = prm.filter + (uint64_t)prevShard * 4;
            if constexpr (TMA_FLUSH) {
                const uint64_t w4[4] = {acc[0], NW > 1 ? acc[NW > 1 ? 1 : 0] : 0, NW > 2 ? acc[NW > 2 ? 2 : 0] : 0,
                                        NW > 3 ? acc[NW > 3 ? 3 : 0] : 0};
                tma_or_sector(dst, w4, flush_slots, n_flushed);
            } else {
#pragma unroll
                for (int q = 0; q < NW; ++q) red_or_64(dst + q, acc[q]);
            }
        }
        if constexpr (TMA_FLUSH) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); // slots intact until read
    } else {
        QueryLane<K, M, S, H, kStreamTPB> ql;
        ql.prologue(W, prm, stage);
        uint32_t res = 0;
        for (int b = 0; b < prm.chunk_blocks; ++b) {
            const uint32_t wnext = __ldg(pw + b + NWIN);
            const uint32_t v16 = __ldg(vw + b);
            uint32_t res16 = 0;
            static_for<0, 16>([&](auto jc) {
                constexpr int J = decltype(jc)::value;
                if (ql.template step<J>(W, prm, stage) == 0) res16 |= 1u << J;
            });
            res16 &= ~v16; // a1: positions without a valid k-mer answer false
#pragma unroll
            for (int i = 0; i + 1 < NWIN; ++i) W[i] = W[i + 1];
            W[NWIN - 1] = wnext;
            res = (res >> 16) | (res16 << 16);
            if (b & 1) {
                const uint64_t wi = (p0 >> 5) + (uint64_t)(b >> 1);
                if (wi < prm.n_bitmap_words) prm.bitmap[wi] = res;
            }
        }
        // the last kLA positions staged look-ahead copies nobody reads; drain them before the next chunk's prologue
        // reuses the same staging slots (two unordered cp.async to one slot could land in either order)
        cp_async_wait<0>();
    }
    } // chunk loop
}

// =============================================================================================
// a2-a6 fused, RECORD MODE (query of short records, e.g. 150-base reads): one thread per record.
// Same per-position arithmetic as the chunk-mode query (QueryLane), but the thread walks exactly its
// record's k-mer start positions, so the K-1 tail positions of every record (20 % of a 150-base
// read at k = 31) cost nothing, record ends need no marking, and the per-record hit count falls out
// of the same registers.  The window is re-aligned to the record start with one funnel shift per
// 16 symbols.  Output: pack_kernel zeroed the bitmap; words that lie wholly inside the record are
// stored, the (at most two) words shared with neighbours are OR-ed in.
// A record longer than rec_limit is not walked here: the thread lists it for stream_long_kernel
// (launched right after), which walks ONLY those records, chunk by chunk; the short records' results
// stand.  Only a batch whose long records overflow the list raises the fallback flag, and the chunk
// kernels, launched behind, then redo the whole batch (they do nothing while the flag is clear).
// =============================================================================================
template <int K, int M, int S, int H>
#ifdef SBF_REC_MAXREG
__global__ void __maxnreg__(SBF_REC_MAXREG) stream_rec_kernel(const StreamParams prm)
#else
__global__ void __launch_bounds__(kRecTPB, SBF_MINB_R) stream_rec_kernel(const StreamParams prm)
#endif
{
    __shared__ uint4 stage[kNS * 2 * kRecTPB];

    const uint64_t r = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= prm.n_rec) return;
    const uint64_t a = __ldg(prm.offsets + r), e = __ldg(prm.offsets + r + 1);
    if (e - a > (uint64_t)prm.rec_limit) {
        // too long for one thread: hand the record to stream_long_kernel as groups of chunks on the batch's 128-position
        // grid.  Only when the list cannot hold them (or there is none) does the flag go up and the chunk kernels redo
        // the whole batch.
        const uint64_t nch = ((e - 1) >> 7) - (a >> 7) + 1;
        const uint64_t ngr = (nch + kLongGroup - 1) / kLongGroup;
        if (prm.long_groups != nullptr && ngr <= (uint64_t)prm.long_cap) {
            const uint32_t base = atomicAdd(prm.fallback + 1, (uint32_t)ngr);
            if ((uint64_t)base + ngr <= (uint64_t)prm.long_cap) {
                for (uint32_t j = 0; j < (uint32_t)ngr; ++j) prm.long_groups[base + j] = make_uint2((uint32_t)r, j);
                if (prm.counts) prm.counts[r] = 0; // stream_long_kernel adds its chunks' hits
                return;
            }
        }
        *prm.fallback = 1;
        return;
    }
    const uint32_t len = (uint32_t)(e - a);
    const uint32_t nk = len >= (uint32_t)K ? len - K + 1 : 0; // k-mer start positions of the record
    if (nk == 0) {
        if (prm.counts) prm.counts[r] = 0;
        return;
    }
    const uint32_t *__restrict__ pw = prm.packed + (a >> 4);
    const uint16_t *__restrict__ vw = prm.vmask + (a >> 4);
    const uint32_t s2 = 2u * (uint32_t)(a & 15), s1 = (uint32_t)(a & 15);
    constexpr int NWIN = kWinOf(K);
    uint32_t rawLast;
    uint32_t W[NWIN];
    {
        uint32_t raw[NWIN + 1];
#pragma unroll
        for (int i = 0; i <= NWIN; ++i) raw[i] = __ldg(pw + i);
#pragma unroll
        for (int i = 0; i < NWIN; ++i) W[i] = __funnelshift_l(raw[i + 1], raw[i], s2);
        rawLast = raw[NWIN];
    }
    uint32_t vcur = (uint32_t)__ldg(vw) | ((uint32_t)__ldg(vw + 1) << 16); // V bits of the symbols from 16*(a>>4) on

    QueryLane<K, M, S, H, kRecTPB> ql;
    ql.prologue(W, prm, stage);

    // result bits leave through a 64-bit buffer aligned to the bitmap's words
    uint64_t rb = 0;
    uint32_t fill = (uint32_t)(a & 31), cnt = 0;
    uint32_t *bw = prm.bitmap + (a >> 5);                      // the bitmap word being filled
    const uint32_t w_shared = (uint32_t)((e >> 5) - (a >> 5)); // words from this index on reach past the record's end
    uint32_t wrel = 0;
    auto emit = [&](uint32_t word) {
        if (wrel == 0 || wrel >= w_shared) { // shared with a neighbouring record (or the first word: a is rarely 32-aligned)
            if (word) atomicOr(bw, word);
        } else {
            *bw = word;
        }
        ++bw;
        ++wrel;
    };

    const uint32_t nblk = (nk + 15) >> 4;
    for (uint32_t b = 0; b < nblk; ++b) {
        const uint32_t rawNext = __ldg(pw + b + NWIN + 1);
        const uint32_t vNext = __ldg(vw + b + 2);
        uint32_t res16 = 0;
        static_for<0, 8>([&](auto jc) {
            constexpr int J = decltype(jc)::value;
            if (ql.template step<J>(W, prm, stage) == 0) res16 |= 1u << J;
        });
        if (16 * b + 8 < nk)
            static_for<8, 16>([&](auto jc) {
                constexpr int J = decltype(jc)::value;
                if (ql.template step<J>(W, prm, stage) == 0) res16 |= 1u << J;
            });
#pragma unroll
        for (int i = 0; i + 1 < NWIN; ++i) W[i] = W[i + 1];
        W[NWIN - 1] = __funnelshift_l(rawNext, rawLast, s2);
        rawLast = rawNext;
        res16 &= ~(vcur >> s1) & 0xFFFFu;   // a1: V bits of these 16 positions (re-aligned like the window)
        vcur = (vcur >> 16) | (vNext << 16);
        if (16 * b + 16 > nk) res16 &= (1u << (nk - 16 * b)) - 1u; // positions past the record's last k-mer
        cnt += __popc(res16);
        rb |= (uint64_t)res16 << fill;
        fill += 16;
        if (fill >= 32) {
            emit((uint32_t)rb);
            rb >>= 32;
            fill -= 32;
        }
    }
    if (rb) emit((uint32_t)rb);
    if (prm.counts) prm.counts[r] = cnt;
}

// =============================================================================================
// a2-a6 fused, the LONG records of a record-mode batch: one CTA per listed group of kLongGroup chunks,
// one thread per chunk of kLongChunk positions on the batch's 128-position grid — the chunk-mode
// query pipeline (QueryLane, 8 blocks of 16), but the result bits are clipped to the record's k-mer
// start positions [a, e-K+1) and OR-ed into the bitmap (pack_kernel zeroed it; the words at the two
// ends are shared with the neighbouring records that stream_rec_kernel answered), and the hits are
// added to the record's count.  The cost follows the long records' symbols only.
// =============================================================================================
template <int K, int M, int S, int H>
__global__ void __launch_bounds__(kStreamTPB, 4) stream_long_kernel(const StreamParams prm)
{
    constexpr int NWIN = kWinOf(K);
    __shared__ uint4 stage[kNS * 2 * kStreamTPB];
    if (*prm.fallback != 0) return; // the list overflowed: the chunk kernels redo the batch
    const uint32_t n_groups = prm.fallback[1];
    for (uint32_t g = blockIdx.x; g < n_groups; g += gridDim.x) {
        const uint2 rj = prm.long_groups[g];
        const uint64_t a = __ldg(prm.offsets + rj.x), e = __ldg(prm.offsets + rj.x + 1);
        const uint64_t lim = e - (uint64_t)(K - 1);                     // one past the record's last k-mer start (e - a > K)
        const uint64_t p0 = ((a >> 7) + (uint64_t)rj.y * kLongGroup + threadIdx.x) << 7;
        uint32_t cnt = 0;
        if (p0 < lim) {
            const uint32_t *__restrict__ pw = prm.packed + (p0 >> 4);
            const uint16_t *__restrict__ vw = prm.vmask + (p0 >> 4);
            uint32_t W[NWIN];
#pragma unroll
            for (int i = 0; i < NWIN; ++i) W[i] = __ldg(pw + i);
            QueryLane<K, M, S, H, kStreamTPB> ql;
            ql.prologue(W, prm, stage);
            uint32_t res = 0;
            for (int b = 0; b < (int)(kLongChunk / 16); ++b) {
                const uint32_t wnext = __ldg(pw + b + NWIN);
                const uint32_t v16 = __ldg(vw + b);
                uint32_t res16 = 0;
                static_for<0, 16>([&](auto jc) {
                    constexpr int J = decltype(jc)::value;
                    if (ql.template step<J>(W, prm, stage) == 0) res16 |= 1u << J;
                });
                res16 &= ~v16; // a1: positions without a valid k-mer answer false
#pragma unroll
                for (int i = 0; i + 1 < NWIN; ++i) W[i] = W[i + 1];
                W[NWIN - 1] = wnext;
                res = (res >> 16) | (res16 << 16);
                if (b & 1) {
                    const uint64_t w0 = p0 + 32ull * (uint64_t)(b >> 1);   // first position of this bitmap word
                    const uint64_t lo = a > w0 ? a : w0, hi = lim < w0 + 32 ? lim : w0 + 32;
                    if (hi > lo) {
                        const uint32_t n = (uint32_t)(hi - lo);
                        const uint32_t word = res & ((n == 32 ? 0xFFFFFFFFu : ((1u << n) - 1u)) << (uint32_t)(lo - w0));
                        if (word) atomicOr(prm.bitmap + (w0 >> 5), word);
                        cnt += __popc(word);
                    }
                }
            }
            cp_async_wait<0>(); // look-ahead copies nobody reads: drained before the next group reuses the slots
        }
        if (prm.counts != nullptr && cnt != 0) atomicAdd(prm.counts + rj.x, cnt);
    }
}

// =============================================================================================
// Runtime-parameter kernel: Alg. 1 / Alg. 2 as printed, one k-mer per thread, everything
// recomputed per k-mer.  Serves every legal (k,m,s,H) that has no
// specialised instance, including H > 10 (A6).  A warp covers 32 consecutive positions, so the
// query result word is one ballot.
// =============================================================================================
__device__ __forceinline__ uint64_t load_kmer(const uint32_t *__restrict__ packed, uint64_t p, int k)
{
    const uint32_t *w = packed + (p >> 4);
    uint32_t a = __ldg(w), b = __ldg(w + 1), c = __ldg(w + 2);
    int sh = 2 * (int)(p & 15);
    uint32_t hi = __funnelshift_l(b, a, sh); // symbols p .. p+15
    uint32_t lo = __funnelshift_l(c, b, sh); // symbols p+16 .. p+31
    uint64_t v = ((uint64_t)hi << 32) | lo;
    return v >> (64 - 2 * k);
}

__device__ __forceinline__ bool kmer_invalid(const uint16_t *__restrict__ vmask, uint64_t p)
{
    return ((__ldg(vmask + (p >> 4)) >> (p & 15)) & 1u) != 0;
}

template <bool INSERT>
__global__ void __launch_bounds__(256) naive_kernel(const NaiveParams np)
{
    const StreamParams &prm = np.sp;
    const int k = np.k, m = np.m, s = np.s, H = np.H;
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; // grid covers a multiple of 32 positions
    bool present = false;
    if (p < prm.n_pos && !kmer_invalid(prm.vmask, p)) {
        const uint64_t v = load_kmer(prm.packed, p, k);
        uint32_t minKey = 0xFFFFFFFFu;
        for (int i = 0; i <= k - m; ++i) { // Alg. 1 l.5-9
            uint64_t x = (v >> (2 * (k - m - i))) & low_mask64(2 * m);
            minKey = min(minKey, g_key(x, m));
        }
        uint64_t *sh = prm.filter + sigma_shard(minKey, prm.shard_shift) * 4;
        uint64_t w[4] = {0, 0, 0, 0};
        if constexpr (!INSERT) ld_shard_256(sh, w);
        uint64_t mk[4] = {0, 0, 0, 0};
        for (int j = 0; j <= k - s; ++j) { // Alg. 1 l.11-14 / Alg. 2 Contains
            uint64_t x = (v >> (2 * (k - s - j))) & low_mask64(2 * s);
            uint64_t h = f_hash(x, s);
            for (int i = 0; i < H; ++i) {
                uint64_t bit = 1ull << bit_pos(h, i, H);
                switch (i & 3) {
                case 0: mk[0] |= bit; break;
                case 1: mk[1] |= bit; break;
                case 2: mk[2] |= bit; break;
                default: mk[3] |= bit; break;
                }
            }
        }
        if constexpr (INSERT) {
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (mk[q]) red_or_64(sh + q, mk[q]);
        } else {
            present = ((mk[0] & ~w[0]) | (mk[1] & ~w[1]) | (mk[2] & ~w[2]) | (mk[3] & ~w[3])) == 0;
        }
    }
    if constexpr (!INSERT) {
        uint32_t word = __ballot_sync(0xFFFFFFFFu, present);
        if ((threadIdx.x & 31) == 0) {
            uint64_t wi = p >> 5;
            if (wi < prm.n_bitmap_words) prm.bitmap[wi] = word;
        }
    }
}

// =============================================================================================
// WIDE runtime-parameter path: the other alphabets of P:139 — protein (26 symbols, 5 bits),
// DNA triplets (64 symbols, 6 bits, three bytes per symbol) — and packed k-mers wider than one 64-bit word (P:153,
// P:435): k * symbol bits <= 128, straight from the ASCII bytes (no pack pass).  Readings A19-A22 of DESIGN.md §3:
//   A19 symbols; triplet symbols sit at multiples of 3 bytes from the record start, windows slide by one symbol
//   A20 the packed k-mer is a 128-bit value, first symbol most significant
//   A21 a window wider than 64 bits is folded before hashing: lo ^ rotl32(hi * 0x9E3779B97F4A7C15); the seeds of g and
//       f are masked to min(window bits, 64)
//   A22 bit index of the result bitmap = BYTE position of the k-mer's first byte
// =============================================================================================
struct WideParams {
    const uint8_t *bases;    // ASCII, all records concatenated
    uint64_t total;          // bytes
    const uint64_t *offsets; // n_rec + 1 (nullptr: one record)
    uint64_t n_rec;
    uint64_t *filter;
    int shard_shift;         // 32 - P
    uint32_t *bitmap;        // query: ceil(total/32) words, all written
    uint64_t n_bitmap_words;
    int k, m, s, H;
    int alphabet;            // 0 DNA, 1 protein, 2 DNA triplet
    int sym_bits, sym_bytes;
    int phase0;              // bytes of the record holding byte 0 that precede the buffer, mod sym_bytes (host-facing chunks)
};

__device__ __forceinline__ int dna_code(uint32_t c)
{
    c &= 0xDFu;
    return c == 'A' ? 0 : c == 'C' ? 1 : c == 'G' ? 2 : c == 'T' ? 3 : -1;
}
#ifdef SBF_DEFINE_AUX_KERNELS
// ---------------------------------------------------------------------------------------------
// wide_tile_kernel, CTA-cooperative.  Done one k-mer per thread, Alg. 1 / Alg. 2 recompute per k-mer the k symbol
// codes, k-m+1 m-mer keys and k-s+1 s-mer hashes (each a 128-bit shift, mask, fold and multiply) and search the
// offsets for the record: ~1000 instructions per k-mer (round 2's first wide_kernel: 6-22 G k-mers/s).  Here a CTA of
// 256 threads takes a tile of 1024 byte positions (+ a 64-byte halo: k * symbol bytes <= 64) through shared memory:
//   A  raw bytes -> code of the symbol STARTING at every byte (0xFF invalid); warp 0 meanwhile finds the record
//      holding the tile's first byte (32-ary search over the offsets) and the CTA lists the record boundaries that
//      fall inside the tile;
//   B  every m-mer key, every s-mer's four sector-word masks and "these k symbols hold an invalid one" ONCE per start
//      byte: a thread rolls the packed windows along five consecutive symbols of one frame (one 128-bit shift-or per
//      symbol instead of m or s);
//   C  one k-mer per thread and byte: validity from the record boundaries, the symbol grid and the rolled invalid
//      flag, minimum of k-m+1 keys, OR of k-s+1 mask quadruples — then the shard update / test of Alg. 1 / Alg. 2.
//      A warp covers 32 consecutive bytes: the query result word is one ballot.
// 2.2-4.9 x the one-k-mer-per-thread form (protein k=12: 51, k=25: 43, triplets k=10: 16, DNA k=63 without a
// specialised instance: 31 G k-mers/s on 60 MB).  A tile with more record boundaries than it has room for (thousands
// of empty records in 1 KiB) looks its records up in global memory instead.
// ---------------------------------------------------------------------------------------------
constexpr int kWtTPB = 256, kWtTile = 1024, kWtHalo = 64, kWtSpan = kWtTile + kWtHalo, kWtStrip = 5; // 218 strips of 5 symbols: one per thread

__device__ __forceinline__ int wide_symbol_smem(const uint8_t *raw, int alphabet)
{
    if (alphabet == 0) return dna_code(raw[0]);
    if (alphabet == 1) {
        const uint32_t c = raw[0] & 0xDFu;
        return (c >= 'A' && c <= 'Z' && (raw[0] & 0x40u)) ? (int)(c - 'A') : -1;
    }
    const int c0 = dna_code(raw[0]), c1 = dna_code(raw[1]), c2 = dna_code(raw[2]);
    return (c0 | c1 | c2) < 0 ? -1 : 16 * c0 + 4 * c1 + c2;
}

// a packed window of up to 128 bits as four 32-bit words (w[3] most significant); symbol widths are below 32 bits
struct Win128 {
    uint32_t w[4];
    __device__ __forceinline__ void clear() { w[0] = w[1] = w[2] = w[3] = 0; }
    __device__ __forceinline__ void push(uint32_t c, int b) // (v << b) | c
    {
        w[3] = __funnelshift_l(w[2], w[3], b);
        w[2] = __funnelshift_l(w[1], w[2], b);
        w[1] = __funnelshift_l(w[0], w[1], b);
        w[0] = (w[0] << b) | c;
    }
    __device__ __forceinline__ void mask(const uint32_t (&m)[4]) { w[0] &= m[0]; w[1] &= m[1]; w[2] &= m[2]; w[3] &= m[3]; }
    __device__ __forceinline__ uint64_t fold() const // A21: lo ^ rotl32(hi * golden)
    {
        const uint64_t lo = ((uint64_t)w[1] << 32) | w[0], hi = ((uint64_t)w[3] << 32) | w[2];
        const uint64_t t = hi * kGold64;
        return lo ^ ((t << 32) | (t >> 32));
    }
};
__device__ __forceinline__ void low_mask128(int nbits, uint32_t (&m)[4])
{
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int r = nbits - 32 * i;
        m[i] = r >= 32 ? 0xFFFFFFFFu : r <= 0 ? 0u : ((1u << r) - 1u);
    }
}

template <bool INSERT, int NB> // NB = bytes per symbol (1: DNA, protein; 3: DNA triplets)
__global__ void __launch_bounds__(kWtTPB) wide_tile_kernel(const WideParams prm)
{
    __shared__ __align__(16) ulonglong2 s_mk01[kWtSpan], s_mk23[kWtSpan]; // one-hot sector words of the s-mer starting at each byte
    __shared__ uint32_t s_gk[kWtSpan];                    // key of the m-mer starting at each byte
    __shared__ uint16_t s_bnd[kWtSpan + 8];               // record boundaries in (t0, t0 + span), relative to t0
    __shared__ uint8_t s_raw[kWtSpan + 8], s_code[kWtSpan + 8];
    __shared__ uint8_t s_kbad[kWtSpan];                   // the k symbols starting at each byte hold an invalid one
    __shared__ uint64_t s_rec0[2];                        // index and start of the record holding byte t0
    __shared__ int s_nbnd;                                // boundaries listed; -1: too many, look records up globally
    __shared__ unsigned s_frames;                         // NB > 1: bit f = some record of the tile has its symbol grid on frame f

    const int k = prm.k, m = prm.m, s = prm.s, H = prm.H, b = prm.sym_bits;
    const int tid = threadIdx.x;
    const uint64_t t0 = (uint64_t)blockIdx.x * kWtTile;

    // ---- A: raw bytes; the first record (warp 0)
    for (int i = tid; i < kWtSpan + 8; i += kWtTPB) {
        const uint64_t q = t0 + (uint64_t)i;
        s_raw[i] = q < prm.total ? __ldg(prm.bases + q) : (uint8_t)0;
    }
    if (tid < 32) {
        uint64_t lo = 0;
        if (prm.offsets != nullptr) {
            uint64_t hi = prm.n_rec; // offsets[lo] <= t0 < offsets[hi]
            while (hi - lo > 1) {
                const uint64_t step = (hi - lo + 32) / 33;
                const uint64_t idx = lo + (uint64_t)(tid + 1) * step;
                const bool le = idx < hi && __ldg(prm.offsets + idx) <= t0;
                const int c = __popc(__ballot_sync(0xFFFFFFFFu, le));
                const uint64_t nhi = c < 32 ? lo + (uint64_t)(c + 1) * step : hi;
                lo += (uint64_t)c * step;
                hi = nhi < hi ? nhi : hi;
            }
        }
        if (tid == 0) {
            s_rec0[0] = lo;
            s_rec0[1] = prm.offsets != nullptr ? __ldg(prm.offsets + lo) : 0;
            s_nbnd = 0;
            s_frames = 0;
        }
    }
    __syncthreads();
    // the boundaries after that record, while they fall inside the tile and its halo
    if (prm.offsets != nullptr) {
        const uint64_t first = s_rec0[0] + 1;
        for (int round = 0;; ++round) {
            const uint64_t idx = first + (uint64_t)round * kWtTPB + tid;
            const uint64_t v = idx <= prm.n_rec ? __ldg(prm.offsets + idx) : ~0ull;
            const bool inside = v < t0 + kWtSpan;
            const int slot = round * kWtTPB + tid;
            if (inside && slot < kWtSpan) s_bnd[slot] = (uint16_t)(v - t0);
            const int n = __syncthreads_count(inside);
            if (tid == 0) s_nbnd = (s_nbnd < 0 || s_nbnd + n > kWtSpan) ? -1 : s_nbnd + n;
            if (n < kWtTPB || (round + 1) * kWtTPB >= kWtSpan + kWtTPB) break;
        }
    }
    for (int i = tid; i < kWtSpan; i += kWtTPB) {
        const int c = wide_symbol_smem(s_raw + i, prm.alphabet);
        s_code[i] = (uint8_t)(c < 0 ? 0xFF : c);
    }
    if (NB > 1) { // which of the NB frames (byte position mod NB inside the tile) carry some record's symbol grid (A19)
        __syncthreads(); // thread 0 wrote s_nbnd after the boundary loop's last barrier: order that write before the reads below
        const int nb_listed = s_nbnd;
        if (nb_listed < 0) {
            if (tid == 0) s_frames = (1u << NB) - 1u;
        } else {
            for (int i = tid; i <= nb_listed; i += kWtTPB) { // record 0 of the tile, then the records starting at the boundaries
                const uint64_t a = i == 0 ? s_rec0[1] : t0 + s_bnd[i - 1];
                const unsigned ph = a == 0 ? (unsigned)prm.phase0 % NB : 0u;
                atomicOr(&s_frames, 1u << (((unsigned)(a % NB) + 2u * NB - ph - (unsigned)(t0 % NB)) % NB));
            }
        }
    }
    __syncthreads();

    // ---- B: m-mer keys, s-mer masks and k-symbol validity, rolled along kWtStrip consecutive symbols of one frame
    {
        const int mbits = m * b < 64 ? m * b : 64, sbits = s * b < 64 ? s * b : 64;
        const uint64_t seedm = kSeedM & low_mask64(mbits), seeds = kSeedS & low_mask64(sbits);
        uint32_t mmask[4], smask[4];
        low_mask128(m * b, mmask);
        low_mask128(s * b, smask);
        const uint64_t kvmask = k < 64 ? ((1ull << k) - 1ull) : ~0ull;
        const int Wd = 64 / H; // bit-slice width (A5); below 6 the salted form (A6)
        constexpr int per_frame = (kWtSpan + NB - 1) / NB;               // symbol starts of one frame inside the span
        constexpr int strips_per_frame = (per_frame + kWtStrip - 1) / kWtStrip;
        auto code_at = [&](int q) -> uint32_t { return q < kWtSpan ? (uint32_t)s_code[q] : 0xFFu; };
        for (int sidx = tid; sidx < strips_per_frame * NB; sidx += kWtTPB) {
            const int phi = sidx / strips_per_frame, j0 = (sidx % strips_per_frame) * kWtStrip; // frame-major: whole warps skip a dead frame
            int q = phi + j0 * NB;
            if (q >= kWtSpan) continue;
            if (NB > 1 && !((s_frames >> phi) & 1u)) continue; // no record of this tile has a k-mer on this frame
            Win128 vm, vs;
            vm.clear(); vs.clear();
            uint64_t inv = 0; // bit i = the symbol i places before the newest of the k-symbol window is invalid
            for (int i = 0; i < k; ++i) {
                const uint32_t c = code_at(q + i * NB);
                if (i < m) vm.push(c & 63u, b);
                if (i < s) vs.push(c & 63u, b);
                inv = (inv << 1) | (uint64_t)(c == 0xFFu);
            }
            for (int j = 0; j < kWtStrip && q < kWtSpan; ++j, q += NB) {
                const uint64_t xm = vm.fold() ^ seedm;
                s_gk[q] = ((uint32_t)xm ^ (uint32_t)(xm >> 32)) * kMultG;
                s_kbad[q] = (uint8_t)((inv & kvmask) != 0);
                const uint64_t xs = vs.fold() ^ seeds;
                uint64_t h = (xs ^ (xs >> 28)) * kMultF;
                h ^= h >> 32;
                uint64_t mk0 = 0, mk1 = 0, mk2 = 0, mk3 = 0;
                if (Wd >= 6) { // A5: hash index i -> bits [i Wd, i Wd + 6) of h, word i mod 4
                    uint64_t hh = h;
                    for (int i = 0; i < H; i += 4) {
                        mk0 |= 1ull << (hh & 63); hh >>= Wd;
                        if (i + 1 < H) { mk1 |= 1ull << (hh & 63); hh >>= Wd; }
                        if (i + 2 < H) { mk2 |= 1ull << (hh & 63); hh >>= Wd; }
                        if (i + 3 < H) { mk3 |= 1ull << (hh & 63); hh >>= Wd; }
                    }
                } else {       // A6: salted upper bits
                    for (int i = 0; i < H; ++i) {
                        const uint64_t bit = 1ull << ((h * ((uint64_t)(2 * i + 1) * kGold64)) >> 58);
                        if ((i & 3) == 0) mk0 |= bit; else if ((i & 3) == 1) mk1 |= bit; else if ((i & 3) == 2) mk2 |= bit; else mk3 |= bit;
                    }
                }
                s_mk01[q] = make_ulonglong2(mk0, mk1);
                s_mk23[q] = make_ulonglong2(mk2, mk3);
                const uint32_t cm = code_at(q + m * NB), cs = code_at(q + s * NB), ck = code_at(q + k * NB);
                vm.push(cm & 63u, b); vm.mask(mmask);
                vs.push(cs & 63u, b); vs.mask(smask);
                inv = (inv << 1) | (uint64_t)(ck == 0xFFu);
            }
        }
    }
    __syncthreads();

    // ---- C: one k-mer per thread and byte
    const int nbnd = s_nbnd;
    const int nkm = k - m, nks = k - s;
    for (int j = 0; j < kWtTile / kWtTPB; ++j) {
        const int pr = j * kWtTPB + tid;
        const uint64_t p = t0 + (uint64_t)pr;
        bool present = false;
        if (!s_kbad[pr]) { // k valid symbols from here on (bytes past the end of the buffer are invalid symbols)
            int e_rel = 0x7FFFFFFF; // end of the record holding p, relative to t0 (no boundary inside the halo: far enough)
            uint64_t a = 0;
            if (prm.offsets != nullptr) {
                if (nbnd >= 0) { // boundaries <= p among the listed ones
                    int lo = 0, hi = nbnd;
                    while (lo < hi) {
                        const int mid = (lo + hi) >> 1;
                        if ((int)s_bnd[mid] <= pr) lo = mid + 1; else hi = mid;
                    }
                    if (lo < nbnd) e_rel = (int)s_bnd[lo];
                    if (NB > 1) a = lo == 0 ? s_rec0[1] : t0 + s_bnd[lo - 1];
                } else {
                    uint64_t lo = 0, hi = prm.n_rec;
                    while (hi - lo > 1) {
                        const uint64_t mid = lo + (hi - lo) / 2;
                        if (__ldg(prm.offsets + mid) <= p) lo = mid; else hi = mid;
                    }
                    a = __ldg(prm.offsets + lo);
                    const uint64_t e = __ldg(prm.offsets + lo + 1);
                    if (e - t0 < 0x7FFFFFFFull) e_rel = (int)(e - t0);
                }
            }
            bool on_grid = true; // A19: symbols sit at multiples of NB bytes from the record start
            if (NB > 1) on_grid = (p - a + (a == 0 ? (uint64_t)prm.phase0 : 0)) % (uint64_t)NB == 0;
            if (on_grid && pr + k * NB <= e_rel) {
                uint32_t minKey = 0xFFFFFFFFu;
                for (int i = 0; i <= nkm; ++i) minKey = min(minKey, s_gk[pr + i * NB]); // Alg. 1 l.5-9
                uint64_t *sh = prm.filter + sigma_shard(minKey, prm.shard_shift) * 4;
                uint64_t w[4] = {0, 0, 0, 0};
                if constexpr (!INSERT) ld_shard_256(sh, w);
                ulonglong2 m01 = make_ulonglong2(0, 0), m23 = make_ulonglong2(0, 0);
                for (int jj = 0; jj <= nks; ++jj) { // Alg. 1 l.11-14 / Alg. 2 Contains
                    const ulonglong2 x = s_mk01[pr + jj * NB], y = s_mk23[pr + jj * NB];
                    m01.x |= x.x; m01.y |= x.y; m23.x |= y.x; m23.y |= y.y;
                }
                if constexpr (INSERT) {
                    if (m01.x) red_or_64(sh + 0, m01.x);
                    if (m01.y) red_or_64(sh + 1, m01.y);
                    if (m23.x) red_or_64(sh + 2, m23.x);
                    if (m23.y) red_or_64(sh + 3, m23.y);
                } else {
                    present = ((m01.x & ~w[0]) | (m01.y & ~w[1]) | (m23.x & ~w[2]) | (m23.y & ~w[3])) == 0;
                }
            }
        }
        if constexpr (!INSERT) {
            const uint32_t word = __ballot_sync(0xFFFFFFFFu, present);
            if ((tid & 31) == 0) {
                const uint64_t wi = p >> 5;
                if (wi < prm.n_bitmap_words) prm.bitmap[wi] = word;
            }
        }
    }
}
#endif // SBF_DEFINE_AUX_KERNELS

// =============================================================================================
// a6: hit counts from the result bitmap.
// =============================================================================================
__device__ __forceinline__ uint32_t popc_range(const uint32_t *__restrict__ bm, uint64_t a, uint64_t e)
{
    // set bits in bit positions [a, e)
    if (a >= e) return 0;
    uint64_t wa = a >> 5, we = (e - 1) >> 5;
    uint32_t first = 0xFFFFFFFFu << (a & 31);
    uint32_t last = 0xFFFFFFFFu >> (31 - ((e - 1) & 31));
    if (wa == we) return __popc(__ldg(bm + wa) & first & last);
    uint32_t c = __popc(__ldg(bm + wa) & first) + __popc(__ldg(bm + we) & last);
    for (uint64_t w = wa + 1; w < we; ++w) c += __popc(__ldg(bm + w));
    return c;
}

#ifdef SBF_DEFINE_AUX_KERNELS
// short records: one thread per record
__global__ void __launch_bounds__(256) count_records_thread_kernel(const uint32_t *__restrict__ bm, const uint64_t *__restrict__ offsets,
                                                                   uint64_t n_rec, uint32_t *__restrict__ counts,
                                                                   const uint32_t *only_if)
{
    if (only_if != nullptr && *only_if == 0) return; // stream_rec_kernel wrote the counts
    for (uint64_t r = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; r < n_rec; r += (uint64_t)gridDim.x * blockDim.x)
        counts[r] = popc_range(bm, offsets[r], offsets[r + 1]);
}

// long records: one CTA per record, grid-stride over records
__global__ void __launch_bounds__(256) count_records_block_kernel(const uint32_t *__restrict__ bm, const uint64_t *__restrict__ offsets,
                                                                  uint64_t n_rec, uint32_t *__restrict__ counts)
{
    __shared__ uint32_t part[8];
    for (uint64_t r = blockIdx.x; r < n_rec; r += gridDim.x) {
        uint64_t a = offsets[r], e = offsets[r + 1];
        uint32_t c = 0;
        // split [a,e) in 32-aligned pieces, one per thread per round
        uint64_t a32 = a & ~31ull;
        for (uint64_t w = a32 + 32ull * threadIdx.x; w < e; w += 32ull * blockDim.x) {
            uint64_t lo = w < a ? a : w, hi = (w + 32 < e) ? w + 32 : e;
            c += popc_range(bm, lo, hi);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xFFFFFFFFu, c, o);
        if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = c;
        __syncthreads();
        if (threadIdx.x == 0) {
            uint32_t t = 0;
            for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += part[i];
            counts[r] = t;
        }
        __syncthreads();
    }
}

// total popcount of n_words words -> *hits (must be zeroed before)
__global__ void __launch_bounds__(256) count_total_kernel(const uint32_t *__restrict__ bm, uint64_t n_words, unsigned long long *hits)
{
    unsigned long long c = 0;
    for (uint64_t w = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; w < n_words; w += (uint64_t)gridDim.x * blockDim.x)
        c += __popc(__ldg(bm + w));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xFFFFFFFFu, c, o);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(hits, c);
}

// host-facing path: offsets of one chunk [a, a+n) of a batch from the batch's offsets (already on the device):
// out = {0, full[0]-a, ..., full[n_inner-1]-a, n}, full pointing at the first boundary inside the chunk
__global__ void __launch_bounds__(256) rebase_offsets_kernel(const uint64_t *__restrict__ full, uint64_t n_inner, uint64_t a, uint64_t n,
                                                             uint64_t *__restrict__ out)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) {
        out[0] = 0;
        out[n_inner + 1] = n;
    }
    if (i < n_inner) out[1 + i] = full[i] - a;
}

// filter |= src  (replica merge)
__global__ void __launch_bounds__(256) or_words_kernel(uint64_t *__restrict__ dst, const uint64_t *__restrict__ src, uint64_t n_words)
{
    uint64_t n2 = n_words / 2;
    ulonglong2 *d2 = reinterpret_cast<ulonglong2 *>(dst);
    const ulonglong2 *s2 = reinterpret_cast<const ulonglong2 *>(src);
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += (uint64_t)gridDim.x * blockDim.x) {
        ulonglong2 a = d2[i], b = s2[i];
        a.x |= b.x; a.y |= b.y;
        d2[i] = a;
    }
}

// filter[range] |= OR over the peers' replicas of the same range, read in place through peer pointers (NVLink P2P / CUDA
// IPC mappings, or other filters on this device): the reduce-scatter step of the replica merge as ONE kernel per
// window — no staging buffer, no separate receive.  src holds up to kMaxPeers device pointers to the START of the range.
constexpr int kMaxPeers = 15;
struct PeerPtrs { const uint64_t *p[kMaxPeers]; };
__global__ void __launch_bounds__(256) or_peers_kernel(uint64_t *__restrict__ dst, PeerPtrs src, int n_src, uint64_t n_words)
{
    const uint64_t n2 = n_words / 2;
    ulonglong2 *d2 = reinterpret_cast<ulonglong2 *>(dst);
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += (uint64_t)gridDim.x * blockDim.x) {
        ulonglong2 a = d2[i];
        for (int j = 0; j < n_src; ++j) {
            const ulonglong2 b = reinterpret_cast<const ulonglong2 *>(src.p[j])[i];
            a.x |= b.x; a.y |= b.y;
        }
        d2[i] = a;
    }
}

#endif // SBF_DEFINE_AUX_KERNELS

} // namespace sbfk

// sbf_device.cuh — device code of the Super Bloom filter hot path (sm_100a).
//
// P:<n> = line n of the paper's extracted text; A<n> = reading n in DESIGN.md §3.
// This file restates the pinned arithmetic on its own; it shares nothing with oracle/.
//
// Kernels
//   pack_kernel        a1  ASCII -> 2-bit words (16 bases / uint32, first base in the top bits)
//                          + "k-mer cannot start here" mask G (1 bit / base)
//   mark_ends_kernel   a1  ORs the record-end bits into G
//   stream_kernel      a2-a6  the fused, thread-serial streaming insert / query kernel
//   naive_kernel       a2-a6  runtime-parameter one-k-mer-per-thread form of Alg. 1/2 (any legal k,m,s,H)
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
#define SBF_Q_LA 3   // query: the minimizer runs this many positions ahead of the bit tests
#endif
#ifndef SBF_Q_PF
#define SBF_Q_PF 3   // query (chunk mode): 0 load at first use, 1 prefetch.global.L2 ahead, 3 cp.async staging in shared memory
#endif
#ifndef SBF_IDP_EXTRACT
#define SBF_IDP_EXTRACT 1 // bit-slice extraction by IDP.4A where the slice is byte aligned (H = 1, 2, 4, 8)
#endif
#ifndef SBF_MINB_I
#define SBF_MINB_I 5 // insert: CTAs per SM the register budget is cut for (5 x 128 threads -> 96 registers)
#endif
#ifndef SBF_MINB_Q
#define SBF_MINB_Q 5 // query: 5 x 128 threads -> 96 registers
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
constexpr int kStreamTPB = 128; // threads per CTA of stream_kernel
constexpr int kPadWords = 16;   // zero / all-invalid words appended to the packed sequence and its mask

struct StreamParams {
    const uint32_t *packed; // 2-bit words, ceil(n_pos/16) + kPadWords
    const uint16_t *gmask;  // one uint16 per packed word: bit j = G[16*word + j]
    uint64_t n_pos;         // symbols in the batch (= k-mer start positions walked)
    uint64_t *filter;       // 4 * numShards sector words
    int shard_shift;        // 32 - P
    uint32_t *bitmap;       // query: ceil(n_pos/32) words
    uint64_t n_bitmap_words;
    // record mode (stream_rec_kernel): one thread per record
    const uint64_t *offsets; // n_rec + 1
    uint64_t n_rec;
    uint32_t *counts;        // nullable: per-record hit counts
    const uint32_t *max_len; // device word written by mark_ends_kernel: longest record of the batch
    uint32_t rec_limit;      // record mode runs iff *max_len <= rec_limit (the chunk kernels run otherwise)
    int chunk_blocks;        // chunk mode: 16-position blocks walked by one thread (2, 4 or 8: small batches use short chunks)
};

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

// =============================================================================================
// a1: pack.  Thread i produces packed words 2i, 2i+1 and their mask words from symbols [32i, 32i+32).
//   code: A=0 C=1 G=2 T=3 (either case, A9); anything else is invalid (code bits arbitrary).
//   B[j] = symbol j invalid or j >= len.   G[j] = B[j] | B[j+1] (k >= 2), = B[j] (k == 1).
//   A k-mer starting at p is valid iff G[p .. p+max(k-1,1)-1] are all 0 once mark_ends_kernel
//   has added F[j] = "a record ends after symbol j" (no k-mer spans records).
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

#ifdef SBF_DEFINE_AUX_KERNELS // non-template kernels: defined in one translation unit (sbf_api.cu)
__global__ void __launch_bounds__(256) pack_kernel(const uint8_t *__restrict__ seq, uint64_t len, uint32_t *__restrict__ packed,
                                                   uint16_t *__restrict__ gmask, uint64_t n_words_total, int k, int aligned16)
{
    // thread i: symbols [32i, 32i+32) -> packed words 2i, 2i+1 (one 8-byte store) and their two mask words (one 4-byte store)
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t b0 = i * 32;
    uint32_t v[8];
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
    uint32_t word[2] = {0, 0}, inv = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
        uint32_t i4;
        const uint32_t c8 = pack4(v[w], i4);
        word[w >> 2] |= c8 << (24 - 8 * (w & 3));
        inv |= i4 << (4 * w);
    }
    // B of the next symbol: first flag of the next lane, or a direct byte load at the warp edge
    uint32_t nxt = __shfl_down_sync(0xFFFFFFFFu, inv & 1u, 1);
    if ((threadIdx.x & 31) == 31) {
        const uint64_t p = b0 + 32;
        uint32_t c = (p < len) ? (uint32_t)seq[p] : (uint32_t)'N';
        c &= 0xDFu;
        nxt = !(c == 'A' || c == 'C' || c == 'G' || c == 'T');
    }
    const uint32_t g = (k >= 2) ? (inv | (inv >> 1) | (nxt << 31)) : inv;
    if (2 * i + 1 < n_words_total) {
        *reinterpret_cast<uint2 *>(packed + 2 * i) = make_uint2(word[0], word[1]);
        *reinterpret_cast<uint32_t *>(gmask + 2 * i) = g;
    } else if (2 * i < n_words_total) {
        packed[2 * i] = word[0];
        gmask[2 * i] = (uint16_t)g;
    }
}

// F bits: a record boundary after symbol offsets[r]-1, r = 1..n_rec  (k >= 2 only); also the longest
// record of the batch -> *max_len (nullable), which selects record mode or chunk mode on the device.
__global__ void __launch_bounds__(256) mark_ends_kernel(const uint64_t *__restrict__ offsets, uint64_t n_rec, uint64_t total,
                                                        uint32_t *gmask32, int k, uint32_t *max_len)
{
    const uint64_t r = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x + 1;
    uint32_t len = 0;
    if (r <= n_rec) {
        const uint64_t e = offsets[r], a = offsets[r - 1];
        const uint64_t l64 = e >= a ? e - a : 0;
        len = l64 > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)l64;
        if (k >= 2 && e != 0 && e <= total) {
            const uint64_t j = e - 1;
            atomicOr(&gmask32[j >> 5], 1u << (j & 31));
        }
    }
    if (max_len != nullptr) {
        // one atomic per warp, and only while it can still raise the maximum (monotone, so the stale read is safe)
        len = __reduce_max_sync(0xFFFFFFFFu, len);
        if ((threadIdx.x & 31) == 0 && len > *reinterpret_cast<volatile uint32_t *>(max_len)) atomicMax(max_len, len);
    }
}

#endif // SBF_DEFINE_AUX_KERNELS

// =============================================================================================
// Window access for stream_kernel.  W[0..3] hold 64 consecutive symbols (W[0] first, first symbol
// in the top bits).  lmer<O,N>(W) = the N-mer starting O symbols into the window, as Sub() of the
// paper's packed k-mer (first base most significant).  All shifts are immediates.
// =============================================================================================
constexpr int kWin = 4; // 32-bit words in the register window

template <int Q, int NB>
__device__ __forceinline__ uint32_t field_win(const uint32_t (&W)[kWin])
{
    // bits [Q, Q+NB) of the window, counted from the least significant bit of W[kWin-1]
    static_assert(Q >= 0 && NB >= 1 && NB <= 32 && Q + NB <= 32 * kWin, "field outside the register window");
    constexpr int idx = Q / 32, sh = Q % 32;
    uint32_t lo = W[kWin - 1 - idx];
    uint32_t v;
    if constexpr (sh == 0) {
        v = lo;
    } else if constexpr (sh + NB <= 32) {
        v = lo >> sh;
    } else {
        v = __funnelshift_r(lo, W[kWin - 2 - idx], sh);
    }
    if constexpr (NB < 32 && !(sh + NB == 32)) v &= (1u << NB) - 1u;
    return v;
}

template <int O, int N>
__device__ __forceinline__ uint64_t lmer(const uint32_t (&W)[kWin])
{
    constexpr int Q = 32 * kWin - 2 * O - 2 * N;
    constexpr int nb = 2 * N;
    uint32_t lo = field_win<Q, (nb < 32 ? nb : 32)>(W);
    uint32_t hi = 0;
    if constexpr (nb > 32) hi = field_win<Q + 32, nb - 32>(W);
    return ((uint64_t)hi << 32) | lo;
}

__device__ __forceinline__ uint32_t min3u(uint32_t a, uint32_t b, uint32_t c) { return min(min(a, b), c); }

// Sliding minimum of the last WN keys, streaming: keys arrive one per step, E = step phase (mod 16
// is all that matters).  Levels c3 = min of the last 3, c9 = min of the last 9; the window of WN is
// covered by two or three overlapping blocks (three-input minimum = VIMNMX3 on sm_100a).
template <int WN>
struct SlidingMin {
    static_assert(WN >= 1 && WN <= 24, "stream kernel supports k-m+1 <= 24");
    uint32_t g[16], c3[16], c9[16];
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
            else return min3u(a9, c9[(E - 9) & 15], c9[(E - (WN - 9)) & 15]);
        }
        return gn;
    }
};

// One-hot sector masks of one s-mer hash: hash index i -> word i mod 4, bit B(h,i) (A5)
template <int OFF>
__device__ __forceinline__ uint64_t onehot_at(uint64_t h)
{
#if SBF_IDP_EXTRACT
    if constexpr (OFF % 8 == 0) {
        // byte-aligned slice: mask all four bytes of the half at once (shared by the other slices of that half), then
        // pick the byte with a byte dot product (IDP.4A runs off the alu pipe that bounds the query kernels)
        const uint32_t half = OFF < 32 ? (uint32_t)h : (uint32_t)(h >> 32);
        const uint32_t b = __dp4a(half & 0x3F3F3F3Fu, 1u << (OFF % 32), 0u);
        return 1ull << b;
    }
#endif
    return 1ull << ((h >> OFF) & 63);
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

// A2 with the shift clamped in hardware (shard_shift = 32 when there is one shard)
__device__ __forceinline__ uint32_t sigma32(uint32_t key, int shard_shift)
{
    uint32_t t = (uint32_t)(((uint64_t)key * kGold64) >> 32);
    return __funnelshift_rc(t, 0u, (uint32_t)shard_shift);
}

// query staging through shared memory (SBF_Q_PF == 3): the 32 bytes of a shard travel global -> shared with two
// 16-byte cp.async (LDGSTS, no register in between) LA positions before the run's first test reads them back.
__device__ __forceinline__ void cp_async_shard(uint4 *smem_lo, uint4 *smem_hi, const uint64_t *g)
{
    uint32_t a = (uint32_t)__cvta_generic_to_shared(smem_lo), b = (uint32_t)__cvta_generic_to_shared(smem_hi);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(a), "l"(g) : "memory");
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(b), "l"(g + 2) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ void prefetch_shard(const uint64_t *p)
{
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}

// =============================================================================================
// a2-a6 fused.  One thread walks kChunk consecutive k-mer start positions p0 .. p0+kChunk-1 of the
// batch, carrying in registers: the 64-symbol window, the sliding-minimum rings (a2), the one-hot
// masks of the last k-s s-mers, and
//   insert: the OR of the current super-k-mer's masks (a5), flushed with one RED.OR.B64 per sector
//           word when the shard (A14) or validity changes;
//   query : the current shard's 256 bits (a6), reloaded when the shard changes; the k-mer's mask
//           K = OR of its k-s+1 s-mer masks is tested with K & ~shard == 0 (Findere rule).
//           The minimizer runs LA positions ahead of the tests so that the shard of an upcoming
//           run can be prefetched long before its first test.
// Each m-mer key and each s-mer hash is computed once per position (not once per k-mer as in
// Alg. 1/2); the result bits are the same because OR/AND do not care about order or repetition.
// =============================================================================================
template <int K, int M, int S, int H, bool INSERT>
__global__ void __launch_bounds__(kStreamTPB, INSERT ? SBF_MINB_I : SBF_MINB_Q) stream_kernel(const StreamParams prm)
{
    constexpr int WN = K - M + 1;
    constexpr int Z = K - S;
    constexpr int NW = H < 4 ? H : 4;
    constexpr int RZ = ring_size(Z);
    constexpr int L = K > 1 ? K - 1 : 1;
    constexpr int LA = INSERT ? 0 : SBF_Q_LA;
    constexpr uint32_t maskL = (L >= 32) ? 0xFFFFFFFFu : ((1u << L) - 1u);
    static_assert(K >= 1 && K <= 32 && M >= 1 && M <= K && S >= 1 && S <= K, "bad k/m/s");
    static_assert(Z <= 16, "stream kernel supports k-s <= 16");
    static_assert(LA >= 0 && LA <= 16 && (LA == 0 || SBF_Q_PF == 3 || 16 % LA == 0), "lookahead must divide 16");

    if constexpr (!INSERT) {
        if (prm.max_len != nullptr && __ldg(prm.max_len) <= prm.rec_limit) return; // stream_rec_kernel did this batch
    }
    // one chunk per thread; the (normally idle) fallback launch behind record mode uses a small grid and strides
    for (uint64_t chunk = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;; chunk += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t p0 = chunk * (uint64_t)(16 * prm.chunk_blocks);
    if (p0 >= prm.n_pos) return;

    const uint32_t *__restrict__ pw = prm.packed + (p0 >> 4);
    const uint16_t *__restrict__ gw = prm.gmask + (p0 >> 4);
    uint32_t W[kWin] = {__ldg(pw), __ldg(pw + 1), __ldg(pw + 2), __ldg(pw + 3)};
    uint32_t glo = (uint32_t)__ldg(gw) | ((uint32_t)__ldg(gw + 1) << 16);
    uint32_t ghi = (uint32_t)__ldg(gw + 2) | ((uint32_t)__ldg(gw + 3) << 16);

    SlidingMin<WN> smin;
#pragma unroll
    for (int i = 0; i < 16; ++i) { smin.g[i] = 0; smin.c3[i] = 0; smin.c9[i] = 0; }
    uint64_t Mh[RZ][NW];
#pragma unroll
    for (int i = 0; i < RZ; ++i)
#pragma unroll
        for (int q = 0; q < NW; ++q) Mh[i][q] = 0;

    // prologue: keys of the first WN-1 m-mers, masks of the first Z s-mers
    static_for<0, WN - 1>([&](auto ec) {
        constexpr int E = decltype(ec)::value;
        (void)smin.template push<E>(g_key(lmer<E, M>(W), M));
    });
    static_for<0, Z>([&](auto ic) {
        constexpr int I = decltype(ic)::value;
        expand_masks<H, NW>(f_hash_c<S>(lmer<I, S>(W)), Mh[I % RZ]);
    });
    uint64_t PB[NW], PC[NW]; // query, Z == 3: ORs of adjacent mask pairs (see the test below)
#pragma unroll
    for (int q = 0; q < NW; ++q) {
        PB[q] = Mh[0][q] | Mh[1 % RZ][q];
        PC[q] = Mh[1 % RZ][q] | Mh[2 % RZ][q];
    }
    // query: shards of the first LA k-mers, prefetched (PF 1/2) or staged in shared memory (PF 3)
    constexpr bool STAGE = !INSERT && SBF_Q_PF == 3;
    constexpr int NS = LA + 1; // staging slots per thread: k-mer q uses slot q mod NS
    static_assert(!STAGE || (LA >= 1 && 16 % NS == 0), "staging needs LA in {1,3,7,15}");
    __shared__ uint4 stage[STAGE ? NS * 2 * kStreamTPB : 1];
    uint32_t kq[LA > 0 ? LA : 1];
    uint32_t laPrev = 0xFFFFFFFFu;
    bool sb[NS]; // sb[q mod NS]: a run starts at k-mer q (its shard is in staging slot q mod NS)
#pragma unroll
    for (int i = 0; i < NS; ++i) sb[i] = false;
    bool laInv = true;
    (void)laPrev; (void)sb; (void)laInv; (void)stage;
    kq[0] = 0;
    static_for<0, LA>([&](auto ec) {
        constexpr int Q = decltype(ec)::value;
        constexpr int E = Q + WN - 1;
        const uint32_t sh = sigma32(smin.template push<E>(g_key(lmer<E, M>(W), M)), prm.shard_shift);
        if constexpr (STAGE) {
            const bool invN = (__funnelshift_r(glo, ghi, Q) & maskL) != 0;
            const bool start = !invN && (laInv || sh != laPrev);
            if (start)
                cp_async_shard(&stage[((Q % NS) * 2) * kStreamTPB + threadIdx.x], &stage[((Q % NS) * 2 + 1) * kStreamTPB + threadIdx.x],
                               prm.filter + (uint64_t)sh * 4);
            cp_async_commit();
            sb[Q % NS] = start;
            laInv = invN;
        } else {
            kq[Q] = sh;
            if (SBF_Q_PF != 0 && (Q == 0 || sh != laPrev)) prefetch_shard(prm.filter + (uint64_t)sh * 4);
        }
        laPrev = sh;
    });

    uint64_t acc[NW];   // insert: OR of the current run's masks
    uint64_t shard[4];  // query: the current shard's sector words
#pragma unroll
    for (int q = 0; q < NW; ++q) acc[q] = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) shard[q] = 0;
    uint32_t prevShard = 0;
    bool prevInval = true; // insert: previous k-mer invalid; query: no shard loaded yet
    uint32_t res = 0;

    for (int b = 0; b < prm.chunk_blocks; ++b) {
        const uint32_t wnext = __ldg(pw + b + 4);
        const uint32_t gnext = __ldg(gw + b + 4);
        uint32_t res16 = 0;
        static_for<0, 16>([&](auto jc) {
            constexpr int J = decltype(jc)::value;
            // a2/a3: key of the newest m-mer of k-mer p+LA (p = p0+16b+J), its window minimum, its shard
            const uint32_t shNew =
                sigma32(smin.template push<J + LA + WN - 1>(g_key(lmer<J + LA + WN - 1, M>(W), M)), prm.shard_shift);
            uint32_t sh = shNew;
            (void)sh;
            if constexpr (STAGE) {
                const bool invN = (__funnelshift_r(glo, ghi, J + LA) & maskL) != 0;
                const bool start = !invN && (laInv || shNew != laPrev);
                if (start)
                    cp_async_shard(&stage[(((J + LA) % NS) * 2) * kStreamTPB + threadIdx.x],
                                   &stage[(((J + LA) % NS) * 2 + 1) * kStreamTPB + threadIdx.x], prm.filter + (uint64_t)shNew * 4);
                cp_async_commit();
                sb[(J + LA) % NS] = start;
                laInv = invN;
                laPrev = shNew;
            } else if constexpr (LA > 0) {
                if (SBF_Q_PF != 0 && shNew != laPrev) prefetch_shard(prm.filter + (uint64_t)shNew * 4);
                laPrev = shNew;
                sh = kq[J % LA];
                kq[J % LA] = shNew;
            }
            // a4: the newest s-mer of k-mer p
            uint64_t Mn[NW];
            expand_masks<H, NW>(f_hash_c<S>(lmer<J + Z, S>(W)), Mn);
            // a1: validity of k-mer p
            const bool inval = (__funnelshift_r(glo, ghi, J) & maskL) != 0;
            if constexpr (INSERT) {
                const bool brk = (sh != prevShard) || (inval != prevInval);
                if (brk) {
                    if (!prevInval) { // a5: flush the finished run
                        uint64_t *dst = prm.filter + (uint64_t)prevShard * 4;
#pragma unroll
                        for (int q = 0; q < NW; ++q) red_or_64(dst + q, acc[q]);
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
            } else {
                if constexpr (STAGE) {
                    if (sb[J % NS]) { // a6: the run starting here: its shard was staged LA positions ago
                        cp_async_wait<LA>();
                        const uint4 lo = stage[((J % NS) * 2) * kStreamTPB + threadIdx.x];
                        const uint4 hi = stage[((J % NS) * 2 + 1) * kStreamTPB + threadIdx.x];
                        shard[0] = ((uint64_t)lo.y << 32) | lo.x; shard[1] = ((uint64_t)lo.w << 32) | lo.z;
                        shard[2] = ((uint64_t)hi.y << 32) | hi.x; shard[3] = ((uint64_t)hi.w << 32) | hi.z;
                    }
                } else {
                    const bool need = !inval && (prevInval || sh != prevShard);
                    if (need) { // a6: fetch the shard of the new run
                        ld_shard_256(prm.filter + (uint64_t)sh * 4, shard);
                        prevShard = sh;
                        prevInval = false;
                    }
                }
                uint64_t miss = 0;
                if constexpr (Z == 3) {
                    // pair ORs: PB = M[t-2]|M[t-3], PC = M[t-1]|M[t-2]; K = (Mn | M[t-1]) | PB
                    uint64_t mq[NW];
#pragma unroll
                    for (int q = 0; q < NW; ++q) {
                        const uint64_t cn = Mn[q] | Mh[(J + 2) % RZ][q];
                        mq[q] = (cn | PB[q]) & ~shard[q];
                        PB[q] = PC[q];
                        PC[q] = cn;
                    }
                    if constexpr (NW == 4) miss = (mq[0] | mq[1] | mq[2]) | mq[3];
                    else
#pragma unroll
                        for (int q = 0; q < NW; ++q) miss |= mq[q];
                } else {
#pragma unroll
                    for (int q = 0; q < NW; ++q) {
                        uint64_t kq_ = Mn[q];
#pragma unroll
                        for (int i = 0; i < Z; ++i) kq_ |= Mh[(J + i) % RZ][q];
                        miss |= kq_ & ~shard[q];
                    }
                }
                if (!inval && miss == 0) res16 |= 1u << J;
            }
#pragma unroll
            for (int q = 0; q < NW; ++q) Mh[(J + Z) % RZ][q] = Mn[q];
        });
        W[0] = W[1]; W[1] = W[2]; W[2] = W[3]; W[3] = wnext;
        glo = (glo >> 16) | (ghi << 16);
        ghi = (ghi >> 16) | (gnext << 16);
        if constexpr (!INSERT) {
            res = (res >> 16) | (res16 << 16);
            if (b & 1) {
                const uint64_t wi = (p0 >> 5) + (uint64_t)(b >> 1);
                if (wi < prm.n_bitmap_words) prm.bitmap[wi] = res;
            }
        }
    }
    if constexpr (INSERT) {
        if (!prevInval) {
            uint64_t *dst = prm.filter + (uint64_t)prevShard * 4;
#pragma unroll
            for (int q = 0; q < NW; ++q) {
                const uint64_t o = acc[q];
                red_or_64(dst + q, o);
            }
        }
    }
    // the last LA positions of a chunk staged look-ahead copies nobody reads; drain them before the next chunk's
    // prologue reuses the same staging slots (two unordered cp.async to one slot could land in either order)
    if constexpr (STAGE) cp_async_wait<0>();
    } // chunk loop
}

// =============================================================================================
// a2-a6 fused, RECORD MODE (query of short records, e.g. 150-base reads): one thread per record.
// Same per-position arithmetic as stream_kernel<..., false> (staged shards, pair-OR masks), but the
// thread walks exactly its record's k-mer start positions, so the K-1 tail positions of every
// record (20 % of a 150-base read at k = 31) cost nothing, and the per-record hit count falls out of
// the same registers.  The window is re-aligned to the record start with one funnel shift per
// 16 symbols.  Output: the bitmap was zeroed by the caller (cudaMemsetAsync); words that lie wholly
// inside the record are stored, the (at most two) words shared with neighbours are OR-ed in.
// Runs only when the longest record of the batch is <= rec_limit (device flag from mark_ends_kernel);
// otherwise every thread exits and the chunk-mode kernels, launched right after, do the work.
// =============================================================================================
template <int K, int M, int S, int H>
__global__ void __launch_bounds__(kStreamTPB, SBF_MINB_R) stream_rec_kernel(const StreamParams prm)
{
    constexpr int WN = K - M + 1;
    constexpr int Z = K - S;
    constexpr int NW = H < 4 ? H : 4;
    constexpr int RZ = ring_size(Z);
    constexpr int L = K > 1 ? K - 1 : 1;
    constexpr int LA = 3, NS = 4;
    constexpr uint32_t maskL = (L >= 32) ? 0xFFFFFFFFu : ((1u << L) - 1u);
    __shared__ uint4 stage[NS * 2 * kStreamTPB];

    if (__ldg(prm.max_len) > prm.rec_limit) return;
    const uint64_t r = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= prm.n_rec) return;
    const uint64_t a = __ldg(prm.offsets + r), e = __ldg(prm.offsets + r + 1);
    const uint32_t len = (uint32_t)(e - a);
    const uint32_t nk = len >= (uint32_t)K ? len - K + 1 : 0; // k-mer start positions of the record
    if (nk == 0) {
        if (prm.counts) prm.counts[r] = 0;
        return;
    }
    const uint32_t *__restrict__ pw = prm.packed + (a >> 4);
    const uint16_t *__restrict__ gw = prm.gmask + (a >> 4);
    const uint32_t s2 = 2u * (uint32_t)(a & 15), s1 = (uint32_t)(a & 15);
    uint32_t rawLast;
    uint32_t W[kWin];
    {
        const uint32_t r0 = __ldg(pw), r1 = __ldg(pw + 1), r2 = __ldg(pw + 2), r3 = __ldg(pw + 3);
        rawLast = __ldg(pw + 4);
        W[0] = __funnelshift_l(r1, r0, s2); W[1] = __funnelshift_l(r2, r1, s2);
        W[2] = __funnelshift_l(r3, r2, s2); W[3] = __funnelshift_l(rawLast, r3, s2);
    }
    uint32_t glo, ghi, gLast; // G bits of positions a.. (bit 0 = position a), re-aligned like the window
    {
        const uint32_t g0 = (uint32_t)__ldg(gw) | ((uint32_t)__ldg(gw + 1) << 16);
        const uint32_t g1 = (uint32_t)__ldg(gw + 2) | ((uint32_t)__ldg(gw + 3) << 16);
        gLast = __ldg(gw + 4);
        glo = __funnelshift_r(g0, g1, s1);
        ghi = __funnelshift_r(g1, gLast, s1);
    }

    SlidingMin<WN> smin;
#pragma unroll
    for (int i = 0; i < 16; ++i) { smin.g[i] = 0; smin.c3[i] = 0; smin.c9[i] = 0; }
    uint64_t Mh[RZ][NW];
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
    uint64_t PB[NW], PC[NW];
#pragma unroll
    for (int q = 0; q < NW; ++q) {
        PB[q] = Mh[0][q] | Mh[1 % RZ][q];
        PC[q] = Mh[1 % RZ][q] | Mh[2 % RZ][q];
    }
    uint32_t laPrev = 0xFFFFFFFFu;
    bool sb[NS], laInv = true;
#pragma unroll
    for (int i = 0; i < NS; ++i) sb[i] = false;
    uint64_t shard[4] = {0, 0, 0, 0};

    // lookahead stage for k-mer q = (block start) + QJ: shard index, run start -> stage the sector
    auto look = [&](auto qc) {
        constexpr int QJ = decltype(qc)::value; // 0 .. 15+LA relative to the current window
        const uint32_t shNew = sigma32(smin.template push<QJ + WN - 1>(g_key(lmer<QJ + WN - 1, M>(W), M)), prm.shard_shift);
        const bool invN = (__funnelshift_r(glo, ghi, QJ) & maskL) != 0;
        const bool start = !invN && (laInv || shNew != laPrev);
        if (start)
            cp_async_shard(&stage[((QJ % NS) * 2) * kStreamTPB + threadIdx.x], &stage[((QJ % NS) * 2 + 1) * kStreamTPB + threadIdx.x],
                           prm.filter + (uint64_t)shNew * 4);
        cp_async_commit();
        sb[QJ % NS] = start;
        laInv = invN;
        laPrev = shNew;
    };
    static_for<0, LA>(look);

    uint32_t res16 = 0;
    auto step = [&](auto jc) {
        constexpr int J = decltype(jc)::value;
        look(std::integral_constant<int, J + LA>{});
        uint64_t Mn[NW];
        expand_masks<H, NW>(f_hash_c<S>(lmer<J + Z, S>(W)), Mn);
        const bool inval = (__funnelshift_r(glo, ghi, J) & maskL) != 0;
        if (sb[J % NS]) {
            cp_async_wait<LA>();
            const uint4 lo = stage[((J % NS) * 2) * kStreamTPB + threadIdx.x];
            const uint4 hi = stage[((J % NS) * 2 + 1) * kStreamTPB + threadIdx.x];
            shard[0] = ((uint64_t)lo.y << 32) | lo.x; shard[1] = ((uint64_t)lo.w << 32) | lo.z;
            shard[2] = ((uint64_t)hi.y << 32) | hi.x; shard[3] = ((uint64_t)hi.w << 32) | hi.z;
        }
        uint64_t miss = 0;
        if constexpr (Z == 3) {
            uint64_t mq[NW];
#pragma unroll
            for (int q = 0; q < NW; ++q) {
                const uint64_t cn = Mn[q] | Mh[(J + 2) % RZ][q];
                mq[q] = (cn | PB[q]) & ~shard[q];
                PB[q] = PC[q];
                PC[q] = cn;
            }
            if constexpr (NW == 4) miss = (mq[0] | mq[1] | mq[2]) | mq[3];
            else
#pragma unroll
                for (int q = 0; q < NW; ++q) miss |= mq[q];
        } else {
#pragma unroll
            for (int q = 0; q < NW; ++q) {
                uint64_t kq_ = Mn[q];
#pragma unroll
                for (int i = 0; i < Z; ++i) kq_ |= Mh[(J + i) % RZ][q];
                miss |= kq_ & ~shard[q];
            }
        }
        if (!inval && miss == 0) res16 |= 1u << J;
#pragma unroll
        for (int q = 0; q < NW; ++q) Mh[(J + Z) % RZ][q] = Mn[q];
    };

    // result bits leave through a 64-bit buffer aligned to the bitmap's words
    uint64_t rb = 0;
    uint32_t fill = (uint32_t)(a & 31), cnt = 0;
    uint64_t wi = a >> 5;
    bool first = true;
    auto emit = [&](uint32_t word) {
        if (first || (wi + 1) * 32 > e) {
            if (word) atomicOr(prm.bitmap + wi, word);
        } else {
            prm.bitmap[wi] = word;
        }
        first = false;
        ++wi;
    };

    const uint32_t nblk = (nk + 15) >> 4;
    for (uint32_t b = 0; b < nblk; ++b) {
        const uint32_t rawNext = __ldg(pw + b + 5);
        const uint32_t gNext = __ldg(gw + b + 5);
        res16 = 0;
        static_for<0, 8>(step);
        if (16 * b + 8 < nk) static_for<8, 16>(step);
        W[0] = W[1]; W[1] = W[2]; W[2] = W[3]; W[3] = __funnelshift_l(rawNext, rawLast, s2);
        rawLast = rawNext;
        // next 16 re-aligned G bits = bits [s1, s1+16) of gLast | gNext << 16
        const uint32_t g16 = (__funnelshift_r(gLast | (gNext << 16), 0u, s1)) & 0xFFFFu;
        glo = (glo >> 16) | (ghi << 16);
        ghi = (ghi >> 16) | (g16 << 16);
        gLast = gNext;
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

__device__ __forceinline__ bool kmer_invalid(const uint16_t *__restrict__ gmask, uint64_t p, int k)
{
    const uint16_t *g = gmask + (p >> 4);
    uint64_t bits = (uint64_t)__ldg(g) | ((uint64_t)__ldg(g + 1) << 16) | ((uint64_t)__ldg(g + 2) << 32);
    int L = k > 1 ? k - 1 : 1;
    return ((bits >> (p & 15)) & low_mask64(L)) != 0;
}

template <bool INSERT>
__global__ void __launch_bounds__(256) naive_kernel(const NaiveParams np)
{
    const StreamParams &prm = np.sp;
    const int k = np.k, m = np.m, s = np.s, H = np.H;
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; // grid covers a multiple of 32 positions
    bool present = false;
    if (p < prm.n_pos && !kmer_invalid(prm.gmask, p, k)) {
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
                                                                   const uint32_t *max_len, uint32_t rec_limit)
{
    if (max_len != nullptr && __ldg(max_len) <= rec_limit) return; // stream_rec_kernel wrote the counts
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

#endif // SBF_DEFINE_AUX_KERNELS

} // namespace sbfk

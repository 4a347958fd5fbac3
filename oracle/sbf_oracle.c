/*
 * sbf_oracle.c — CPU oracle (see sbf_oracle.h: TEST INFRASTRUCTURE, NOT PRODUCT).
 *
 * Plain, slow, per-k-mer restatement of PAPER.md Alg. 1 / Alg. 2.  Every k-mer
 * is packed from scratch, all k-m+1 m-mers and k-s+1 s-mers are re-hashed, no
 * state is carried between k-mers.  P:<n> = /root/reference/PAPER.md line n.
 * A<n> = reading n in DESIGN.md §3 (where the paper gives no constants/rules).
 */
#include "sbf_oracle.h"

#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- pinned constants (A1, A2, A4, A6) ---- */
#define SEED_M   0x5851F42D4C957F2Dull
#define MULT_G   0x9E3779B1u
#define GOLD64   0x9E3779B97F4A7C15ull
#define SEED_S   0x2545F4914F6CDD1Dull
#define MULT_F   0xD6E8FEB86659FD93ull

static uint64_t low_bits(int nbits) { return nbits >= 64 ? ~0ull : ((1ull << nbits) - 1); }

/* A9: case-insensitive ACGT are the valid symbols; 2-bit codes A=0 C=1 G=2 T=3 (2 bits/base) */
int sbfo_code(unsigned char c)
{
    switch (c) {
    case 'A': case 'a': return 0;
    case 'C': case 'c': return 1;
    case 'G': case 'g': return 2;
    case 'T': case 't': return 3;
    default: return -1;
    }
}

/* Subwindow(packed, i, len) of Alg. 1 l.7 / l.12: first base most significant */
uint64_t sbfo_sub(uint64_t v, int k, int i, int len)
{
    return (v >> (2 * (k - len - i))) & low_bits(2 * len);
}

/* A1: "lightweight multiplicative hash" -> 32-bit order key */
uint32_t sbfo_g(int m, uint64_t x)
{
    x ^= SEED_M & low_bits(2 * m);
    uint32_t y = (uint32_t)x ^ (uint32_t)(x >> 32);
    return y * MULT_G;
}

/* A2: minimizer key -> shard in [0, 2^P) (power-of-two shard count, no division) */
uint64_t sbfo_sigma(uint32_t key, int P)
{
    uint64_t t = ((uint64_t)key * GOLD64) >> 32;
    return t >> (32 - P);
}

/* A4: "stronger mix with an additional xorshift" */
uint64_t sbfo_f(int s, uint64_t x)
{
    x ^= SEED_S & low_bits(2 * s);
    uint64_t h = (x ^ (x >> 28)) * MULT_F;
    return h ^ (h >> 32);
}

/* A5 (bit-slicing) for 64/H >= 6; A6 (salt fallback) otherwise */
int sbfo_bitpos(uint64_t h, int i, int H)
{
    int W = 64 / H;
    if (W >= 6)
        return (int)((h >> (i * W)) & 63);
    return (int)((h * ((uint64_t)(2 * i + 1) * GOLD64)) >> 58);
}

sbfo_t *sbfo_create(int k, int m, int s, int H, uint64_t num_bits)
{
    if (k < 1 || k > 32 || m < 1 || m > k || s < 1 || s > k || H < 1 || H > 32 || num_bits < 1)
        return NULL;
    uint64_t need = (num_bits + 255) / 256;      /* shards of 256 bits */
    uint64_t shards = 1;
    int P = 0;
    while (shards < need) { shards <<= 1; ++P; } /* rounded up to a power of two (A8) */
    if (P > 32) return NULL;
    sbfo_t *f = (sbfo_t *)calloc(1, sizeof(*f));
    if (!f) return NULL;
    f->k = k; f->m = m; f->s = s; f->H = H; f->P = P; f->num_shards = shards;
    f->alphabet = SBFO_DNA; f->sym_bits = 2; f->sym_bytes = 1; f->wide = 0;
    f->words = (uint64_t *)calloc(shards * 4, sizeof(uint64_t));
    if (!f->words) { free(f); return NULL; }
    return f;
}

void sbfo_destroy(sbfo_t *f) { if (f) { free(f->words); free(f); } }
void sbfo_clear(sbfo_t *f) { memset(f->words, 0, f->num_shards * 4 * sizeof(uint64_t)); }
uint64_t sbfo_num_shards(const sbfo_t *f) { return f->num_shards; }
const uint64_t *sbfo_words(const sbfo_t *f) { return f->words; }

/* ValidKmer + PackKmer (Alg. 1 l.3-4; shift-and-OR).
 * The k-mer at p exists iff p + k <= L and is valid iff all k symbols are ACGT (A9). */
int sbfo_pack_kmer(const sbfo_t *f, const uint8_t *rec, uint64_t L, uint64_t p, uint64_t *v)
{
    if (p + (uint64_t)f->k > L) return 0;
    uint64_t x = 0;
    for (int i = 0; i < f->k; ++i) {
        int c = sbfo_code(rec[p + i]);
        if (c < 0) return 0;
        x = (x << 2) | (uint64_t)c;
    }
    *v = x;
    return 1;
}

/* Alg. 1 l.5-9: minimum hash over all k-m+1 m-mer windows */
uint32_t sbfo_min_key(const sbfo_t *f, uint64_t v)
{
    uint32_t min_hash = 0xFFFFFFFFu;
    for (int i = 0; i <= f->k - f->m; ++i) {
        uint32_t h = sbfo_g(f->m, sbfo_sub(v, f->k, i, f->m));
        if (h < min_hash) min_hash = h;
    }
    return min_hash;
}

/* Alg. 1 l.10 with the A2 remix in place of the literal low bits */
uint64_t sbfo_shard_of(const sbfo_t *f, uint64_t v)
{
    return sbfo_sigma(sbfo_min_key(f, v), f->P);
}

/* Alg. 1 l.11-14: the four sector-word masks of one k-mer.
 * Hash index i -> sector i mod 4. */
static void kmer_masks(const sbfo_t *f, uint64_t v, uint64_t w[4])
{
    w[0] = w[1] = w[2] = w[3] = 0;
    for (int j = 0; j <= f->k - f->s; ++j) {
        uint64_t s_hash = sbfo_f(f->s, sbfo_sub(v, f->k, j, f->s));
        for (int i = 0; i < f->H; ++i)
            w[i % 4] |= 1ull << sbfo_bitpos(s_hash, i, f->H);
    }
}

void sbfo_insert_kmer(sbfo_t *f, uint64_t v)
{
    uint64_t w[4];
    uint64_t shard = sbfo_shard_of(f, v);
    kmer_masks(f, v, w);
    for (int q = 0; q < 4; ++q)                 /* Alg. 1 l.23-27 */
        f->words[shard * 4 + q] |= w[q];
}

/* Alg. 2 Contains: every s-mer, every hash, its bit must be set */
int sbfo_contains_kmer(const sbfo_t *f, uint64_t v)
{
    const uint64_t *words = f->words + sbfo_shard_of(f, v) * 4;
    int present = 1;
    for (int j = 0; j <= f->k - f->s; ++j) {
        uint64_t s_hash = sbfo_f(f->s, sbfo_sub(v, f->k, j, f->s));
        for (int h = 0; h < f->H; ++h) {
            int sector = h % 4;
            int bit_pos = sbfo_bitpos(s_hash, h, f->H);
            present = present && ((words[sector] >> bit_pos) & 1);
        }
    }
    return present;
}

/* Records are independent; no k-mer spans two records (A11). */
static uint64_t wide_insert_records(sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec, int mt);
static uint64_t wide_query_records(const sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec,
                                   uint32_t *bitmap, uint32_t *hit_counts, int mt);
static uint64_t wide_count_valid(const sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec);

uint64_t sbfo_insert_records(sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec)
{
    if (f->wide) return wide_insert_records(f, bases, offsets, n_rec, 0);
    uint64_t n_valid = 0;
    for (uint64_t r = 0; r < n_rec; ++r) {
        const uint8_t *rec = bases + offsets[r];
        uint64_t L = offsets[r + 1] - offsets[r];
        for (uint64_t p = 0; p + (uint64_t)f->k <= L; ++p) {
            uint64_t v;
            if (sbfo_pack_kmer(f, rec, L, p, &v)) { sbfo_insert_kmer(f, v); ++n_valid; }
        }
    }
    return n_valid;
}

uint64_t sbfo_query_records(const sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec,
                            uint32_t *bitmap, uint32_t *hit_counts)
{
    if (f->wide) return wide_query_records(f, bases, offsets, n_rec, bitmap, hit_counts, 0);
    uint64_t total = offsets[n_rec], n_valid = 0;
    memset(bitmap, 0, ((total + 31) / 32) * sizeof(uint32_t));
    for (uint64_t r = 0; r < n_rec; ++r) {
        const uint8_t *rec = bases + offsets[r];
        uint64_t L = offsets[r + 1] - offsets[r];
        uint32_t hits = 0;
        for (uint64_t p = 0; p + (uint64_t)f->k <= L; ++p) {
            uint64_t v;
            if (!sbfo_pack_kmer(f, rec, L, p, &v)) continue;      /* invalid -> false */
            ++n_valid;
            if (sbfo_contains_kmer(f, v)) {
                uint64_t g = offsets[r] + p;                      /* bit index = global base position */
                bitmap[g >> 5] |= 1u << (g & 31);
                ++hits;
            }
        }
        if (hit_counts) hit_counts[r] = hits;
    }
    return n_valid;
}

uint64_t sbfo_count_valid_kmers(const sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec)
{
    if (f->wide) return wide_count_valid(f, bases, offsets, n_rec);
    uint64_t n_valid = 0;
    for (uint64_t r = 0; r < n_rec; ++r) {
        const uint8_t *rec = bases + offsets[r];
        uint64_t L = offsets[r + 1] - offsets[r], v;
        for (uint64_t p = 0; p + (uint64_t)f->k <= L; ++p)
            n_valid += (uint64_t)sbfo_pack_kmer(f, rec, L, p, &v);
    }
    return n_valid;
}

/* ------------------------------------------------------------------------
 * Multi-core drivers: the same per-k-mer functions, positions split in
 * chunks of 2^16 global base positions (a multiple of 32, so bitmap words are
 * never shared between chunks).  Insert uses atomic fetch-OR.
 * ------------------------------------------------------------------------ */
#define MT_CHUNK 65536ull

static uint64_t record_of(const uint64_t *offsets, uint64_t n_rec, uint64_t g)
{
    /* last r with offsets[r] <= g (skips empty records) */
    uint64_t lo = 0, hi = n_rec;             /* invariant: offsets[lo] <= g < offsets[hi] */
    while (hi - lo > 1) {
        uint64_t mid = lo + (hi - lo) / 2;
        if (offsets[mid] <= g) lo = mid; else hi = mid;
    }
    return lo;
}

uint64_t sbfo_insert_records_mt(sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec)
{
    if (f->wide) return wide_insert_records(f, bases, offsets, n_rec, 1);
    uint64_t total = offsets[n_rec], n_valid = 0;
    int64_t nchunks = (int64_t)((total + MT_CHUNK - 1) / MT_CHUNK);
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : n_valid)
    for (int64_t c = 0; c < nchunks; ++c) {
        uint64_t g0 = (uint64_t)c * MT_CHUNK, g1 = g0 + MT_CHUNK;
        if (g1 > total) g1 = total;
        uint64_t r = record_of(offsets, n_rec, g0);
        for (uint64_t g = g0; g < g1; ++g) {
            while (g >= offsets[r + 1]) ++r;
            uint64_t v, w[4];
            if (!sbfo_pack_kmer(f, bases + offsets[r], offsets[r + 1] - offsets[r], g - offsets[r], &v)) continue;
            ++n_valid;
            uint64_t shard = sbfo_shard_of(f, v);
            kmer_masks(f, v, w);
            for (int q = 0; q < 4; ++q)
                if (w[q]) __atomic_fetch_or(&f->words[shard * 4 + q], w[q], __ATOMIC_RELAXED);
        }
    }
    return n_valid;
}

uint64_t sbfo_query_records_mt(const sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec,
                               uint32_t *bitmap, uint32_t *hit_counts)
{
    if (f->wide) return wide_query_records(f, bases, offsets, n_rec, bitmap, hit_counts, 1);
    uint64_t total = offsets[n_rec], n_valid = 0;
    int64_t nchunks = (int64_t)((total + MT_CHUNK - 1) / MT_CHUNK);
    memset(bitmap, 0, ((total + 31) / 32) * sizeof(uint32_t));
    if (hit_counts) memset(hit_counts, 0, n_rec * sizeof(uint32_t));
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : n_valid)
    for (int64_t c = 0; c < nchunks; ++c) {
        uint64_t g0 = (uint64_t)c * MT_CHUNK, g1 = g0 + MT_CHUNK;
        if (g1 > total) g1 = total;
        uint64_t r = record_of(offsets, n_rec, g0);
        for (uint64_t g = g0; g < g1; ++g) {
            while (g >= offsets[r + 1]) ++r;
            uint64_t v;
            if (!sbfo_pack_kmer(f, bases + offsets[r], offsets[r + 1] - offsets[r], g - offsets[r], &v)) continue;
            ++n_valid;
            if (sbfo_contains_kmer(f, v)) {
                bitmap[g >> 5] |= 1u << (g & 31);
                if (hit_counts) __atomic_fetch_add(&hit_counts[r], 1u, __ATOMIC_RELAXED);
            }
        }
    }
    return n_valid;
}

/* Test scaffolding: per global base position, the min key / shard / validity the per-k-mer functions give. */
uint64_t sbfo_trace_records(const sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec,
                            uint32_t *min_key, uint64_t *shard, uint8_t *valid)
{
    uint64_t total = offsets[n_rec], n_valid = 0;
    int64_t nchunks = (int64_t)((total + MT_CHUNK - 1) / MT_CHUNK);
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : n_valid)
    for (int64_t c = 0; c < nchunks; ++c) {
        uint64_t g0 = (uint64_t)c * MT_CHUNK, g1 = g0 + MT_CHUNK;
        if (g1 > total) g1 = total;
        uint64_t r = record_of(offsets, n_rec, g0);
        for (uint64_t g = g0; g < g1; ++g) {
            while (g >= offsets[r + 1]) ++r;
            uint64_t v;
            int ok = sbfo_pack_kmer(f, bases + offsets[r], offsets[r + 1] - offsets[r], g - offsets[r], &v);
            if (valid) valid[g] = (uint8_t)ok;
            if (min_key) min_key[g] = ok ? sbfo_min_key(f, v) : 0;
            if (shard) shard[g] = ok ? sbfo_shard_of(f, v) : 0;
            n_valid += (uint64_t)ok;
        }
    }
    return n_valid;
}

/* ========================================================================
 * Wide path (readings A19-A22 in DESIGN.md §3): the alphabets of P:139 and
 * packed k-mers wider than one 64-bit word ("for DNA this is possible
 * for k <= 32"; "wider packed representations, such as multiword").
 * The same Alg. 1 / Alg. 2, one k-mer at a time, on a 128-bit packed value.
 * ======================================================================== */
typedef unsigned __int128 u128;

/* A19: DNA = ACGT, either case, 2 bits.  Protein = the 26 letters, either case, 5 bits, code = letter - 'A'.
 * DNA triplet = three consecutive DNA bases, 6 bits, code = 16 c0 + 4 c1 + c2 ("64 symbols, 6 bits, multi-byte"). */
int sbfo_symbol_code(int alphabet, const uint8_t *p)
{
    if (alphabet == SBFO_DNA) return sbfo_code(p[0]);
    if (alphabet == SBFO_PROTEIN) {
        unsigned char c = p[0];
        if (c >= 'a' && c <= 'z') c = (unsigned char)(c - 'a' + 'A');
        return (c >= 'A' && c <= 'Z') ? c - 'A' : -1;
    }
    int c0 = sbfo_code(p[0]), c1 = sbfo_code(p[1]), c2 = sbfo_code(p[2]);
    if (c0 < 0 || c1 < 0 || c2 < 0) return -1;
    return 16 * c0 + 4 * c1 + c2;
}

/* A21: a window of more than 64 bits enters the (64-bit) hashes folded: lo XOR the golden-ratio multiple of hi,
 * rotated by 32.  A window of at most 64 bits has hi = 0 and is passed through unchanged. */
uint64_t sbfo_fold64(uint64_t hi, uint64_t lo)
{
    uint64_t t = hi * GOLD64;
    return lo ^ ((t << 32) | (t >> 32));
}

sbfo_t *sbfo_create_ex(int k, int m, int s, int H, uint64_t num_bits, int alphabet)
{
    int bits = alphabet == SBFO_DNA ? 2 : alphabet == SBFO_PROTEIN ? 5 : alphabet == SBFO_TRIPLET ? 6 : 0;
    if (!bits || k < 1 || k * bits > 128 || m < 1 || m > k || s < 1 || s > k || H < 1 || H > 32 || num_bits < 1) return NULL;
    if (alphabet == SBFO_DNA && k <= 32) return sbfo_create(k, m, s, H, num_bits);
    sbfo_t *f = sbfo_create(1, 1, 1, H, num_bits);          /* geometry (A8) as in the narrow path */
    if (!f) return NULL;
    f->k = k; f->m = m; f->s = s;
    f->alphabet = alphabet; f->sym_bits = bits; f->sym_bytes = alphabet == SBFO_TRIPLET ? 3 : 1; f->wide = 1;
    return f;
}

void sbfo_force_wide(sbfo_t *f, int on) { f->wide = on ? 1 : (f->alphabet != SBFO_DNA || f->k > 32); }

/* ValidKmer + PackKmer (Alg. 1 l.3-4): shift by the symbol width and OR ("left-shift by the alphabet symbol
 * width, OR in the new trailing symbol").  Triplet symbols sit at multiples of three bytes from the record start
 * ("alignment padding to symbolWidth boundaries"), so a k-mer exists only at such a byte. */
int sbfo_pack_kmer_w(const sbfo_t *f, const uint8_t *rec, uint64_t L, uint64_t p, uint64_t *hi, uint64_t *lo)
{
    if (p % (uint64_t)f->sym_bytes != 0) return 0;
    if (p + (uint64_t)f->k * (uint64_t)f->sym_bytes > L) return 0;
    u128 x = 0;
    for (int i = 0; i < f->k; ++i) {
        int c = sbfo_symbol_code(f->alphabet, rec + p + (uint64_t)i * (uint64_t)f->sym_bytes);
        if (c < 0) return 0;
        x = (x << f->sym_bits) | (u128)(unsigned)c;
    }
    *hi = (uint64_t)(x >> 64);
    *lo = (uint64_t)x;
    return 1;
}

/* Subwindow(packed, i, len): len symbols starting i symbols into the k-mer, first symbol most significant */
uint64_t sbfo_sub_w(const sbfo_t *f, uint64_t hi, uint64_t lo, int i, int len)
{
    u128 v = ((u128)hi << 64) | lo;
    int nbits = len * f->sym_bits;
    u128 w = v >> ((f->k - len - i) * f->sym_bits);
    if (nbits < 128) w &= (((u128)1) << nbits) - 1;
    return sbfo_fold64((uint64_t)(w >> 64), (uint64_t)w);
}

/* g and f of a window of nbits bits (A1, A4 with the seed masked to the window width, at most 64 bits) */
static uint32_t g_bits(int nbits, uint64_t x)
{
    x ^= SEED_M & low_bits(nbits);
    uint32_t y = (uint32_t)x ^ (uint32_t)(x >> 32);
    return y * MULT_G;
}
static uint64_t f_bits(int nbits, uint64_t x)
{
    x ^= SEED_S & low_bits(nbits);
    uint64_t h = (x ^ (x >> 28)) * MULT_F;
    return h ^ (h >> 32);
}

uint32_t sbfo_min_key_w(const sbfo_t *f, uint64_t hi, uint64_t lo)
{
    uint32_t min_hash = 0xFFFFFFFFu;
    for (int i = 0; i <= f->k - f->m; ++i) {                         /* Alg. 1 l.5-9 */
        uint32_t h = g_bits(f->m * f->sym_bits, sbfo_sub_w(f, hi, lo, i, f->m));
        if (h < min_hash) min_hash = h;
    }
    return min_hash;
}

uint64_t sbfo_shard_of_w(const sbfo_t *f, uint64_t hi, uint64_t lo)
{
    return sbfo_sigma(sbfo_min_key_w(f, hi, lo), f->P);
}

static void kmer_masks_w(const sbfo_t *f, uint64_t hi, uint64_t lo, uint64_t w[4])
{
    w[0] = w[1] = w[2] = w[3] = 0;
    for (int j = 0; j <= f->k - f->s; ++j) {                         /* Alg. 1 l.11-14 */
        uint64_t s_hash = f_bits(f->s * f->sym_bits, sbfo_sub_w(f, hi, lo, j, f->s));
        for (int i = 0; i < f->H; ++i)
            w[i % 4] |= 1ull << sbfo_bitpos(s_hash, i, f->H);
    }
}

void sbfo_insert_kmer_w(sbfo_t *f, uint64_t hi, uint64_t lo)
{
    uint64_t w[4];
    uint64_t shard = sbfo_shard_of_w(f, hi, lo);
    kmer_masks_w(f, hi, lo, w);
    for (int q = 0; q < 4; ++q) f->words[shard * 4 + q] |= w[q];
}

int sbfo_contains_kmer_w(const sbfo_t *f, uint64_t hi, uint64_t lo)
{
    const uint64_t *words = f->words + sbfo_shard_of_w(f, hi, lo) * 4;
    int present = 1;
    for (int j = 0; j <= f->k - f->s; ++j) {                         /* Alg. 2 Contains */
        uint64_t s_hash = f_bits(f->s * f->sym_bits, sbfo_sub_w(f, hi, lo, j, f->s));
        for (int h = 0; h < f->H; ++h)
            present = present && ((words[h % 4] >> sbfo_bitpos(s_hash, h, f->H)) & 1);
    }
    return present;
}

/* Record drivers of the wide path: every BYTE position p of every record is a candidate k-mer start (a triplet k-mer
 * exists only where p is a multiple of 3); bit index of the query bitmap = global byte position (A22). */
static uint64_t wide_insert_records(sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec, int mt)
{
    uint64_t n_valid = 0;
    int64_t n = (int64_t)n_rec;
    (void)mt;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : n_valid) if (mt)
    for (int64_t r = 0; r < n; ++r) {
        const uint8_t *rec = bases + offsets[r];
        uint64_t L = offsets[r + 1] - offsets[r];
        for (uint64_t p = 0; p < L; ++p) {
            uint64_t hi, lo, w[4];
            if (!sbfo_pack_kmer_w(f, rec, L, p, &hi, &lo)) continue;
            ++n_valid;
            uint64_t shard = sbfo_shard_of_w(f, hi, lo);
            kmer_masks_w(f, hi, lo, w);
            for (int q = 0; q < 4; ++q)
                if (w[q]) __atomic_fetch_or(&f->words[shard * 4 + q], w[q], __ATOMIC_RELAXED);
        }
    }
    return n_valid;
}

static uint64_t wide_query_records(const sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec,
                                   uint32_t *bitmap, uint32_t *hit_counts, int mt)
{
    uint64_t total = offsets[n_rec], n_valid = 0;
    int64_t n = (int64_t)n_rec;
    (void)mt;
    memset(bitmap, 0, ((total + 31) / 32) * sizeof(uint32_t));
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : n_valid) if (mt)
    for (int64_t r = 0; r < n; ++r) {
        const uint8_t *rec = bases + offsets[r];
        uint64_t L = offsets[r + 1] - offsets[r];
        uint32_t hits = 0;
        for (uint64_t p = 0; p < L; ++p) {
            uint64_t hi, lo;
            if (!sbfo_pack_kmer_w(f, rec, L, p, &hi, &lo)) continue;
            ++n_valid;
            if (sbfo_contains_kmer_w(f, hi, lo)) {
                uint64_t g = offsets[r] + p;
                __atomic_fetch_or(&bitmap[g >> 5], 1u << (g & 31), __ATOMIC_RELAXED);   /* records may share a word */
                ++hits;
            }
        }
        if (hit_counts) hit_counts[r] = hits;
    }
    return n_valid;
}

static uint64_t wide_count_valid(const sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec)
{
    uint64_t n_valid = 0;
    for (uint64_t r = 0; r < n_rec; ++r) {
        uint64_t L = offsets[r + 1] - offsets[r], hi, lo;
        for (uint64_t p = 0; p < L; ++p) n_valid += (uint64_t)sbfo_pack_kmer_w(f, bases + offsets[r], L, p, &hi, &lo);
    }
    return n_valid;
}

int sbfo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * seqgen.c — seeded synthetic DNA workloads (sequences, N runs, repeats, reads).
 *
 * Input generation only: this file holds none of the Super Bloom filter's
 * arithmetic (no k-mer packing, no minimizer/s-mer hashing, no filter access).
 * It serves both the CPU oracle's tests and the CUDA path's tests/bench, so the
 * two sides see byte-identical inputs.  The recipes (what each config is made
 * of) are stated in DESIGN.md "Input recipe"; they stand in for the paper's
 * C. elegans / T2T-CHM13 references (§V-A), which are not
 * available offline.
 *
 * All randomness is one counter-based generator sg_rnd(seed, stream, index):
 * any element can be produced independently, so generation is OpenMP-parallel
 * and position-addressable (tests re-derive e.g. which read bases were mutated).
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>
#include <stdlib.h>

#ifdef _OPENMP
#include <omp.h>
#endif

static inline uint64_t mix64(uint64_t z)
{
    z ^= z >> 33; z *= 0xFF51AFD7ED558CCDull;
    z ^= z >> 33; z *= 0xC4CEB9FE1A85EC53ull;
    z ^= z >> 33;
    return z;
}

/* counter-based generator: 64 uniform bits for (seed, stream, index) */
uint64_t sg_rnd(uint64_t seed, uint64_t stream, uint64_t index)
{
    uint64_t a = mix64(seed + 0x9E3779B97F4A7C15ull * (stream + 1));
    return mix64(a ^ mix64(index + 0xD1B54A32D192ED03ull));
}

/* uniform double in [0,1) */
static inline double u01(uint64_t r) { return (double)(r >> 11) * (1.0 / 9007199254740992.0); }
/* uniform integer in [0, n) (n < 2^32 is exact enough: 64-bit multiply-high) */
static inline uint64_t below(uint64_t r, uint64_t n) { return (uint64_t)(((__uint128_t)r * n) >> 64); }

static const char ACGT[4] = { 'A', 'C', 'G', 'T' };

enum { ST_BASE = 0, ST_CTX = 1, ST_TABLE = 2, ST_REP = 3, ST_NRUN = 4, ST_READ_POS = 5,
       ST_READ_BASE = 6, ST_READ_SUB = 7, ST_FAM = 8, ST_FAMCOPY = 9, ST_RECLEN = 10 };

/* i.i.d. uniform A/C/G/T (config 1; also the "uniform random" reads) */
void sg_uniform(uint64_t seed, uint8_t *out, uint64_t n)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < (int64_t)n; ++i)
        out[i] = ACGT[sg_rnd(seed, ST_BASE, (uint64_t)i) >> 62];
}

/*
 * Order-`order` Markov chain (order <= 8).  The transition table has 4^order
 * contexts; each context's distribution is the GC-targeted base distribution
 * (A,T: (1-gc)/2; C,G: gc/2) with every weight multiplied by a seeded factor
 * in [0.5, 1.5) and renormalised.  To keep generation parallel the chain is
 * restarted every SG_CHUNK bases from a seeded context.
 */
#define SG_CHUNK 65536ull

void sg_markov(uint64_t seed, int order, double gc, uint8_t *out, uint64_t n)
{
    const uint32_t nctx = 1u << (2 * order);
    uint64_t *thr = (uint64_t *)malloc((size_t)nctx * 3 * sizeof(uint64_t));
    const double base_w[4] = { (1 - gc) / 2, gc / 2, gc / 2, (1 - gc) / 2 };
    for (uint32_t c = 0; c < nctx; ++c) {
        double w[4], tot = 0;
        for (int b = 0; b < 4; ++b) {
            w[b] = base_w[b] * (0.5 + u01(sg_rnd(seed, ST_TABLE, (uint64_t)c * 4 + b)));
            tot += w[b];
        }
        double acc = 0;
        for (int b = 0; b < 3; ++b) {
            acc += w[b] / tot;
            thr[(size_t)c * 3 + b] = (uint64_t)(acc * 18446744073709551615.0);
        }
    }
    const uint64_t nchunks = (n + SG_CHUNK - 1) / SG_CHUNK;
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t ch = 0; ch < (int64_t)nchunks; ++ch) {
        uint64_t lo = (uint64_t)ch * SG_CHUNK, hi = lo + SG_CHUNK;
        if (hi > n) hi = n;
        uint32_t ctx = (uint32_t)(sg_rnd(seed, ST_CTX, (uint64_t)ch) & (nctx - 1));
        for (uint64_t i = lo; i < hi; ++i) {
            uint64_t r = sg_rnd(seed, ST_BASE, i);
            const uint64_t *t = thr + (size_t)ctx * 3;
            int b = (r >= t[0]) + (r >= t[1]) + (r >= t[2]);
            out[i] = ACGT[b];
            ctx = ((ctx << 2) | (uint32_t)b) & (nctx - 1);
        }
    }
    free(thr);
}

static inline uint8_t substitute(uint8_t c, uint64_t r)
{
    /* replace an ACGT base by one of the other three; leave anything else alone */
    int b;
    switch (c) { case 'A': b = 0; break; case 'C': b = 1; break; case 'G': b = 2; break;
                 case 'T': b = 3; break; default: return c; }
    return ACGT[(b + 1 + (int)below(r, 3)) & 3];
}

/*
 * Config 2: `n_rep` repeats; repeat j copies len_j in [len_lo, len_hi] bases
 * from a random source offset to a random target offset, each copied base
 * substituted with probability `div`.  Applied in order j = 0.. (sequential:
 * later repeats may copy from earlier ones, as real nested repeats do).
 */
void sg_plant_copies(uint64_t seed, uint8_t *seq, uint64_t n, uint32_t n_rep,
                     uint64_t len_lo, uint64_t len_hi, double div)
{
    const uint64_t thresh = (uint64_t)(div * 18446744073709551615.0);
    for (uint32_t j = 0; j < n_rep; ++j) {
        uint64_t len = len_lo + below(sg_rnd(seed, ST_REP, (uint64_t)j * 4 + 0), len_hi - len_lo + 1);
        if (len > n) len = n;
        uint64_t src = below(sg_rnd(seed, ST_REP, (uint64_t)j * 4 + 1), n - len + 1);
        uint64_t dst = below(sg_rnd(seed, ST_REP, (uint64_t)j * 4 + 2), n - len + 1);
        uint8_t *tmp = (uint8_t *)malloc(len);
        memcpy(tmp, seq + src, len);
        for (uint64_t i = 0; i < len; ++i) {
            uint64_t r = sg_rnd(seed, ST_REP + 100 + j, i * 2);
            if (r < thresh) tmp[i] = substitute(tmp[i], sg_rnd(seed, ST_REP + 100 + j, i * 2 + 1));
        }
        memcpy(seq + dst, tmp, len);
        free(tmp);
    }
}

/*
 * Config 4: interspersed repeat families.  Family f has a seeded uniform
 * consensus of length fam_len[f]; copies are written at seeded positions until
 * the family has covered its share of `frac` * n bases; every copy has its own
 * divergence drawn uniformly from [div_lo, div_hi].
 */
void sg_plant_families(uint64_t seed, uint8_t *seq, uint64_t n, uint32_t n_fam,
                       const uint64_t *fam_len, double frac, double div_lo, double div_hi)
{
    for (uint32_t f = 0; f < n_fam; ++f) {
        uint64_t L = fam_len[f];
        if (L == 0 || L > n) continue;
        uint8_t *cons = (uint8_t *)malloc(L);
        for (uint64_t i = 0; i < L; ++i) cons[i] = ACGT[sg_rnd(seed, ST_FAM + 1000 * (f + 1), i) >> 62];
        uint64_t copies = (uint64_t)(frac * (double)n / (double)n_fam / (double)L);
#pragma omp parallel for schedule(dynamic, 64)
        for (int64_t c = 0; c < (int64_t)copies; ++c) {
            uint64_t base = ((uint64_t)f << 40) + (uint64_t)c * 4;
            /* slot the copies so that parallel writers never overlap */
            uint64_t slot = n / copies, off = 0;
            if (slot > L) off = below(sg_rnd(seed, ST_FAMCOPY, base + 0), slot - L + 1);
            uint64_t dst = (uint64_t)c * slot + off;
            if (dst + L > n) continue;
            double div = div_lo + (div_hi - div_lo) * u01(sg_rnd(seed, ST_FAMCOPY, base + 1));
            uint64_t thresh = (uint64_t)(div * 18446744073709551615.0);
            uint64_t cstream = ST_FAMCOPY + 1 + (uint64_t)f * 0x100000000ull + (uint64_t)c;
            for (uint64_t i = 0; i < L; ++i) {
                uint8_t b = cons[i];
                if (sg_rnd(seed, cstream, i * 2) < thresh) b = substitute(b, sg_rnd(seed, cstream, i * 2 + 1));
                seq[dst + i] = b;
            }
        }
        free(cons);
    }
}

/* Config 3: `n_runs` runs of 'N', lengths uniform in [len_lo, len_hi], random positions */
void sg_plant_n_runs(uint64_t seed, uint8_t *seq, uint64_t n, uint32_t n_runs,
                     uint64_t len_lo, uint64_t len_hi)
{
    for (uint32_t j = 0; j < n_runs; ++j) {
        uint64_t len = len_lo + below(sg_rnd(seed, ST_NRUN, (uint64_t)j * 2), len_hi - len_lo + 1);
        if (len > n) len = n;
        uint64_t pos = below(sg_rnd(seed, ST_NRUN, (uint64_t)j * 2 + 1), n - len + 1);
        memset(seq + pos, 'N', len);
    }
}

/* start of sampled read `r` in a sequence of n bases (r even) */
uint64_t sg_read_start(uint64_t seed, uint64_t n, uint32_t read_len, uint64_t r)
{
    return below(sg_rnd(seed, ST_READ_POS, r), n - read_len + 1);
}

/* 1 if base `i` of sampled read `r` is substituted */
int sg_read_is_sub(uint64_t seed, double sub_rate, uint32_t read_len, uint64_t r, uint32_t i)
{
    const uint64_t thresh = (uint64_t)(sub_rate * 18446744073709551615.0);
    return sg_rnd(seed, ST_READ_SUB, r * read_len + i) < thresh;
}

/*
 * Reads [first, first + n_reads) of fixed length, written back to back.
 * Even global index: sampled from `seq` at sg_read_start with i.i.d.
 * substitutions at `sub_rate` ('N' stays 'N').  Odd index: uniform random ACGT.
 */
void sg_reads(uint64_t seed, const uint8_t *seq, uint64_t n, uint64_t first, uint64_t n_reads,
              uint32_t read_len, double sub_rate, uint8_t *out)
{
    const uint64_t thresh = (uint64_t)(sub_rate * 18446744073709551615.0);
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < (int64_t)n_reads; ++q) {
        uint64_t r = first + (uint64_t)q;
        uint8_t *o = out + (uint64_t)q * read_len;
        if ((r & 1) == 0 && seq != NULL && n >= read_len) {
            uint64_t st = sg_read_start(seed, n, read_len, r);
            for (uint32_t i = 0; i < read_len; ++i) {
                uint8_t b = seq[st + i];
                uint64_t ctr = r * read_len + i;
                if (sg_rnd(seed, ST_READ_SUB, ctr) < thresh) b = substitute(b, sg_rnd(seed, ST_READ_BASE, ctr));
                o[i] = b;
            }
        } else {
            for (uint32_t i = 0; i < read_len; ++i)
                o[i] = ACGT[sg_rnd(seed, ST_READ_BASE, r * read_len + i) >> 62];
        }
    }
}

/*
 * Config 4: n_rec record lengths, each drawn uniformly from [lo, hi] and then
 * scaled so they sum to `total`; offsets[0..n_rec] written (offsets[0] = 0).
 */
void sg_record_offsets(uint64_t seed, uint64_t total, uint32_t n_rec, uint64_t lo, uint64_t hi,
                       uint64_t *offsets)
{
    double *w = (double *)malloc(n_rec * sizeof(double)), tot = 0;
    for (uint32_t r = 0; r < n_rec; ++r) {
        w[r] = (double)lo + (double)(hi - lo) * u01(sg_rnd(seed, ST_RECLEN, r));
        tot += w[r];
    }
    offsets[0] = 0;
    double acc = 0;
    for (uint32_t r = 0; r < n_rec; ++r) {
        acc += w[r];
        offsets[r + 1] = (r + 1 == n_rec) ? total : (uint64_t)(acc / tot * (double)total);
    }
    free(w);
}

int sg_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

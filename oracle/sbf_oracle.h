/*
 * sbf_oracle.h — CPU oracle for the Super Bloom filter insert/query path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call this.
 * It shares no code with the CUDA path (paper_2606_24417_b200/csrc) and neither
 * includes the other.
 *
 * It is the plain definition of what the path computes, written from
 * /root/reference/PAPER.md (cited as P:<line>) in the paper's order and
 * notation, one k-mer at a time, with no rolling state, blocking or fusion:
 *   Alg. 1  insert      Alg. 2  query / Contains
 *   §II-B-1      minimizer   §II-B-2      Findere rule
 *   §IV-B   layout      §IV-G   bit-slicing, hashes
 * Where the paper is silent (hash constants, shard mapping, edge rules) it
 * follows the readings A1-A18 listed in DESIGN.md §3.
 *
 * Parity pins (tests/test_oracle_pins.py, tests/test_oracle_wide_pins.py,
 * tests/golden/): every function here is pinned; nothing is "parity unpinned".
 */
#ifndef SBF_ORACLE_H
#define SBF_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sbfo {
    int k, m, s, H;
    int P;                 /* log2(num_shards) */
    uint64_t num_shards;   /* next power of two >= ceil(num_bits/256) */
    uint64_t *words;       /* num_shards * 4 sector words, shard-major */
    /* wide path (A19-A22): other alphabets and k-mers wider than 64 bits */
    int alphabet;          /* SBFO_DNA / SBFO_PROTEIN / SBFO_TRIPLET */
    int sym_bits;          /* 2 / 5 / 6 bits per symbol */
    int sym_bytes;         /* 1 / 1 / 3 input bytes per symbol ("multi-byte") */
    int wide;              /* 1: the record drivers take the 128-bit path */
} sbfo_t;

enum { SBFO_DNA = 0, SBFO_PROTEIN = 1, SBFO_TRIPLET = 2 };

/* --- the pinned primitives (A1, A2, A4, A5, A6, A9) --- */
int      sbfo_code(unsigned char c);                 /* A,C,G,T (any case) -> 0..3, else -1 */
uint64_t sbfo_sub(uint64_t v, int k, int i, int len);/* Sub(v,i,len): len-mer at offset i of a packed k-mer */
uint32_t sbfo_g(int m, uint64_t x);                  /* minimizer order key of an m-mer */
uint64_t sbfo_sigma(uint32_t key, int P);            /* minimizer key -> shard index */
uint64_t sbfo_f(int s, uint64_t x);                  /* s-mer hash */
int      sbfo_bitpos(uint64_t h, int i, int H);      /* B(h,i): bit 0..63 inside sector word i mod 4 */

/* --- filter object --- */
sbfo_t  *sbfo_create(int k, int m, int s, int H, uint64_t num_bits);   /* NULL on bad parameters */
void     sbfo_destroy(sbfo_t *f);
void     sbfo_clear(sbfo_t *f);
uint64_t sbfo_num_shards(const sbfo_t *f);
const uint64_t *sbfo_words(const sbfo_t *f);

/* --- one k-mer (Alg. 1 / Alg. 2 bodies) --- */
/* packs the k-mer starting at p of a record of length L; returns 1 if it exists and is valid */
int      sbfo_pack_kmer(const sbfo_t *f, const uint8_t *rec, uint64_t L, uint64_t p, uint64_t *v);
uint32_t sbfo_min_key(const sbfo_t *f, uint64_t v);
uint64_t sbfo_shard_of(const sbfo_t *f, uint64_t v);
void     sbfo_insert_kmer(sbfo_t *f, uint64_t v);
int      sbfo_contains_kmer(const sbfo_t *f, uint64_t v);

/* --- record batches: the definition, single-threaded --- */
/* offsets[n_rec+1], offsets[0]=0; record r = bases[offsets[r] .. offsets[r+1]) */
uint64_t sbfo_insert_records(sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec);
/* bitmap: ceil(total/32) words, bit p = k-mer starting at global base p is valid and reported present;
 * hit_counts (nullable): per-record popcount.  Returns the number of valid k-mers. */
uint64_t sbfo_query_records(const sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec,
                            uint32_t *bitmap, uint32_t *hit_counts);
uint64_t sbfo_count_valid_kmers(const sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec);

/* --- wide path: any alphabet of P:139, packed k-mer up to 128 bits (k * sym_bits <= 128), readings A19-A22.
 * Same Alg. 1 / Alg. 2, one k-mer at a time; a packed value is the pair (hi, lo), first symbol most significant.
 * The record drivers above call these when f->wide is set (sbfo_create_ex sets it for a non-DNA alphabet or
 * k > 32; sbfo_force_wide lets a test run DNA k <= 32 through this path to pin it against the narrow one). --- */
sbfo_t  *sbfo_create_ex(int k, int m, int s, int H, uint64_t num_bits, int alphabet);
void     sbfo_force_wide(sbfo_t *f, int on);
/* code of the symbol whose first byte is p[0] (sym_bytes bytes are read), or -1 (A19) */
int      sbfo_symbol_code(int alphabet, const uint8_t *p);
/* fold of a window wider than 64 bits to the 64-bit value the hashes take (A21); identity when hi == 0 */
uint64_t sbfo_fold64(uint64_t hi, uint64_t lo);
/* packs the k-mer whose first BYTE is rec[p]; returns 1 if it exists and is valid (triplets: p % 3 == 0 too, A19) */
int      sbfo_pack_kmer_w(const sbfo_t *f, const uint8_t *rec, uint64_t L, uint64_t p, uint64_t *hi, uint64_t *lo);
/* Sub(v, i, len) of a packed k-mer (i, len in symbols), folded to 64 bits */
uint64_t sbfo_sub_w(const sbfo_t *f, uint64_t hi, uint64_t lo, int i, int len);
uint32_t sbfo_min_key_w(const sbfo_t *f, uint64_t hi, uint64_t lo);
uint64_t sbfo_shard_of_w(const sbfo_t *f, uint64_t hi, uint64_t lo);
void     sbfo_insert_kmer_w(sbfo_t *f, uint64_t hi, uint64_t lo);
int      sbfo_contains_kmer_w(const sbfo_t *f, uint64_t hi, uint64_t lo);

/* --- the same per-k-mer functions driven over all host cores (OpenMP).  Legal because OR is
 * order independent (pin P6); tests check the result equals the single-threaded one. --- */
uint64_t sbfo_insert_records_mt(sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec);
uint64_t sbfo_query_records_mt(const sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec,
                               uint32_t *bitmap, uint32_t *hit_counts);
/* test scaffolding: per global base position the min key / shard / validity (any pointer may be NULL) */
uint64_t sbfo_trace_records(const sbfo_t *f, const uint8_t *bases, const uint64_t *offsets, uint64_t n_rec,
                            uint32_t *min_key, uint64_t *shard, uint8_t *valid);
int      sbfo_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif

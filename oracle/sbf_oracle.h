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
 * Parity pins (tests/test_oracle_pins.py, tests/golden/): every function here
 * is pinned; nothing is "parity unpinned".
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
} sbfo_t;

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

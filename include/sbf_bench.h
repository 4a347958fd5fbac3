/*
 * sbf_bench.h — C ABI of libsbf_bench_b200.so: measurement and test hooks, NOT part of the product boundary
 * (include/sbf.h, libsbf_b200.so).  Loaded by bench.py, `python -m paper_2606_24417_b200.ceilings` and the tests only.
 * Status codes are sbf.h's.  Plain pointers and sizes; d_* device, h_* host, all owned by the caller.
 */
#ifndef SBF_BENCH_H
#define SBF_BENCH_H

#include "sbf.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Measured ceilings of the device ("measure ... before quoting a denominator").  Not part of the
 * path; bench.py calls them in the same run as the kernels it times and reports the rooflines against them.
 *
 * sbf_ceiling_pipe_rate — issue rate of one SM sub-partition for a fixed instruction mix, in 1e9 warp instructions
 *   per second, counted in SASS (each loop body is N x one instruction; tests/test_ceilings_sass.py checks the
 *   disassembly) and timed with CUDA events; divide by the SM clock sampled during the call for a per-clock rate.
 *   mode < sbf_ceiling_pipe_modes(); sbf_ceiling_pipe_mode_name(mode) names the mix, e.g. "LOP3" (alu pipe), "IMAD"
 *   (fma pipe), "LOP3:IMAD 3:1".  iters = loop iterations of 256 instructions per warp (2^16 runs ~70 ms).
 *   *clock64_mhz (nullable) = rate of the in-kernel clock64() counter during the run (not the SM clock on this driver).
 * sbf_ceiling_random_sector — random 32-byte-sector accesses per second (in 1e9/s) over a zeroed scratch array of
 *   array_bytes (rounded down to a power of two), allocated and freed inside the call.  mode 0: 4 x red.or.b64 per
 *   sector (the insert kernel's flush), 1: 1 x red.or.b64, 2: one 256-bit ld.global.nc, 3: 2 x 16-byte cp.async into
 *   shared memory, 4: one 32-byte cp.reduce.async.bulk .or.b64 (TMA reduction), 5: mode 2 with the .L2::64B
 *   prefetch-size hint, 6: mode 3 with the .L2::64B hint (the query kernels' staging, exactly), 7: one plain 256-bit
 *   st.global of the whole sector (no fetch needed).
 * Both synchronise the device.
 */
int sbf_ceiling_pipe_modes(void);
const char *sbf_ceiling_pipe_mode_name(int mode);
int sbf_ceiling_pipe_rate(int mode, int iters, double *g_warp_inst_per_s_per_smsp, double *clock64_mhz);
int sbf_ceiling_random_sector(int mode, uint64_t array_bytes, double *g_accesses_per_s);

/*
 * sbf_bench_pack — row a1 on its own: runs pack_kernel over d_seq[0 .. len) exactly as the insert /
 * query calls launch it (this library carries its own compiled copy of the same source) and copies the first n_words
 * 2-bit packed words (16 symbols each, first symbol in the top bits) and their validity masks (bit j of mask w = no
 * valid k-mer starts at symbol 16 w + j) to the host.  n_words <= ceil(len/16) + 16.  Allocates and frees its own
 * scratch; synchronises.
 */
int sbf_bench_pack(const char *d_seq, uint64_t len, int k, uint32_t *h_words, uint16_t *h_mask, uint64_t n_words);

#ifdef __cplusplus
}
#endif
#endif /* SBF_BENCH_H */

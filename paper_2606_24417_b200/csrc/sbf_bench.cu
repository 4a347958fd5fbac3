// sbf_bench.cu — libsbf_bench_b200.so (include/sbf_bench.h): measurement and test hooks kept OUT of the product library.
//
// Measured ceilings of the device the rooflines are quoted against ("measure ...
// before quoting a denominator").  Not part of the hot path: bench.py calls these two entry points in the same run,
// on the same box and clocks as the kernels it times, and writes the results into its JSON line.
//
//   sbf_ceiling_pipe_rate      issue rate of one SM sub-partition (SMSP) for a fixed instruction mix, in WARP
//                              INSTRUCTIONS PER SECOND, counted in SASS: every loop body below is N x one inline-PTX
//                              instruction that ptxas maps 1:1 to the SASS opcode named in kPipeModeName
//                              (tests/test_ceilings_sass.py disassembles the object and counts them), timed with CUDA
//                              events.  The caller divides by the SM clock it samples during the run (bench.py: NVML);
//                              the in-kernel clock64() delta is returned as well, but on this driver that counter does
//                              not tick at the SM clock (it gave 1.58 warp instructions per "cycle" per SMSP).
//   sbf_ceiling_random_sector  random 32-byte-sector accesses per second over an array of a given size, with exactly
//                              the access the fused kernels make (4 x RED.OR.B64 per sector; 2 x 16-byte cp.async; ...)
#include "../../include/sbf_bench.h"

#define SBF_DEFINE_AUX_KERNELS // the copy of pack_kernel that sbf_bench_pack launches
#include "sbf_device.cuh"

#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>

namespace {

constexpr int kPipeChains = 8;   // independent dependency chains per thread (latency 4 / issue interval 2 needs >= 2)
constexpr int kPipeUnroll = 32;  // groups of kPipeChains instructions per loop iteration (256 per iteration: loop control < 2 %)
constexpr int kPipeTPB = 256;    // 8 warps per CTA
constexpr int kPipeCTAsPerSM = 4; // 32 warps per SM = 8 per SMSP, all resident at once (one wave)

// One instruction of the mix on chain c.  MODE: see kPipeModeName.
template <int MODE>
__device__ __forceinline__ void pipe_op(uint32_t (&r)[kPipeChains], int c, int u, uint32_t k0, uint32_t k1)
{
    // which opcode this slot gets: 0 LOP3, 1 IMAD, 2 SHF, 3 IDP.4A, 4 IMAD.HI, 5 PRMT
    int op;
    const int slot = u * kPipeChains + c;
    if (MODE == 0) op = 0;
    else if (MODE == 1) op = 1;
    else if (MODE == 2) op = 2;
    else if (MODE == 3) op = (slot & 1) ? 1 : 0;            // LOP3 : IMAD = 1 : 1
    else if (MODE == 4) op = (slot & 3) == 3 ? 1 : 0;       // 3 : 1
    else if (MODE == 5) op = (slot & 7) == 7 ? 1 : 0;       // 7 : 1
    else if (MODE == 6) op = (slot & 1) ? 2 : 0;            // LOP3 : SHF = 1 : 1 (same pipe)
    else if (MODE == 7) op = 3;
    else if (MODE == 8) op = (slot & 1) ? 3 : 0;            // LOP3 : IDP.4A = 1 : 1
    else if (MODE == 9) op = 4;
    else if (MODE == 10) op = (slot & 1) ? 4 : 0;           // LOP3 : IMAD.HI = 1 : 1
    else if (MODE == 11) op = 5;
    else op = (slot & 3) == 3 ? 4 : 0;                      // LOP3 : IMAD.HI = 3 : 1
    uint32_t &x = r[c];
    if (op == 0) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x) : "r"(k0), "r"(k1));
    else if (op == 1) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(x) : "r"(k0), "r"(k1));
    else if (op == 2) asm volatile("shf.r.wrap.b32 %0, %0, %1, %2;" : "+r"(x) : "r"(k0), "r"(k1));
    else if (op == 3) asm volatile("dp4a.u32.u32 %0, %0, %1, %2;" : "+r"(x) : "r"(k0), "r"(k1));
    else if (op == 4) asm volatile("mad.hi.u32 %0, %0, %1, %2;" : "+r"(x) : "r"(k0), "r"(k1));
    else asm volatile("prmt.b32 %0, %0, %1, %2;" : "+r"(x) : "r"(k0), "r"(k1));
}

template <int MODE>
__global__ void __launch_bounds__(kPipeTPB) pipe_rate_kernel(uint32_t *sink, int iters, uint32_t seed, long long *cycles)
{
    uint32_t r[kPipeChains];
#pragma unroll
    for (int c = 0; c < kPipeChains; ++c) r[c] = threadIdx.x * 2654435761u + seed * (c + 1);
    const uint32_t k0 = seed | 5u, k1 = (seed << 7) | 3u;
    __syncthreads();
    const long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < kPipeUnroll; ++u)
#pragma unroll
            for (int c = 0; c < kPipeChains; ++c) pipe_op<MODE>(r, c, u, k0, k1);
    }
    const long long t1 = clock64();
    uint32_t acc = 0;
#pragma unroll
    for (int c = 0; c < kPipeChains; ++c) acc ^= r[c];
    if (acc == 0x12345u) sink[0] = acc;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

const char *const kPipeModeName[] = {"LOP3", "IMAD", "SHF", "LOP3:IMAD 1:1", "LOP3:IMAD 3:1", "LOP3:IMAD 7:1",
                                     "LOP3:SHF 1:1", "IDP.4A", "LOP3:IDP.4A 1:1", "IMAD.HI", "LOP3:IMAD.HI 1:1", "PRMT",
                                     "LOP3:IMAD.HI 3:1"};
constexpr int kPipeModes = 13;

__device__ __forceinline__ uint64_t mix64(uint64_t x)
{
    x ^= x >> 33; x *= 0xff51afd7ed558ccdULL; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ULL; x ^= x >> 33;
    return x;
}

// MODE 0: 4 x red.or.b64 to the four words of one random sector (what the insert kernel issues per run)
//      1: 1 x red.or.b64
//      2: one 256-bit ld.global.nc of a random sector
//      3: 2 x 16-byte cp.async.cg into shared memory, read back (what the query kernels issue per run)
//      4: one 32-byte cp.reduce.async.bulk .or.b64 from shared memory (TMA reduction) per random sector
//      5: mode 2 with the .L2::64B prefetch-size hint (a miss pulls 64 B from DRAM instead of 128 B)
//      6: mode 3 with the .L2::64B hint (exactly what the query kernels issue per run)
//      7: one plain 256-bit st.global of a whole random sector (a write needs no fetch: one DRAM transaction)
constexpr int kRandTPB = 128;
template <int MODE>
__global__ void __launch_bounds__(kRandTPB) random_sector_kernel(uint64_t *arr, uint64_t sector_mask, uint32_t per_thread, uint64_t *sink)
{
    constexpr int kSlots = 8; // staged sectors in flight per thread (the query kernels keep up to kLA + 1 = 8)
    __shared__ __align__(16) uint64_t stage[(MODE == 3 || MODE == 6) ? kSlots : 2][kRandTPB][4];
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint64_t acc = 0;
    for (uint32_t i = 0; i < per_thread; ++i) {
        const uint64_t h = mix64(t * per_thread + i + 1);
        uint64_t *p = arr + (h & sector_mask) * 4;
        const uint64_t v = 1ull << (h >> 58);
        if (MODE == 0) {
#pragma unroll
            for (int q = 0; q < 4; ++q) asm volatile("red.global.or.b64 [%0], %1;" ::"l"(p + q), "l"(v) : "memory");
        } else if (MODE == 1) {
            asm volatile("red.global.or.b64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
        } else if (MODE == 2) {
            uint64_t w0, w1, w2, w3;
            asm volatile("ld.global.nc.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(w0), "=l"(w1), "=l"(w2), "=l"(w3) : "l"(p));
            acc += w0 ^ w1 ^ w2 ^ w3;
        } else if (MODE == 7) {
            asm volatile("st.global.v4.u64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(v), "l"(v << 1), "l"(v >> 1), "l"(v | 1) : "memory");
        } else if (MODE == 5) {
            uint64_t w0, w1, w2, w3;
            asm volatile("ld.global.nc.L2::64B.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(w0), "=l"(w1), "=l"(w2), "=l"(w3) : "l"(p));
            acc += w0 ^ w1 ^ w2 ^ w3;
        } else if (MODE == 6) {
            const uint32_t s0 = (uint32_t)__cvta_generic_to_shared(&stage[i % kSlots][threadIdx.x][0]);
            asm volatile("cp.async.cg.shared.global.L2::64B [%0], [%1], 16;" ::"r"(s0), "l"(p) : "memory");
            asm volatile("cp.async.cg.shared.global.L2::64B [%0], [%1], 16;" ::"r"(s0 + 16), "l"(p + 2) : "memory");
            asm volatile("cp.async.commit_group;" ::: "memory");
            asm volatile("cp.async.wait_group 7;" ::: "memory");
            acc += stage[(i + 1) % kSlots][threadIdx.x][0] ^ stage[(i + 1) % kSlots][threadIdx.x][3];
        } else if (MODE == 3) {
            const uint32_t s0 = (uint32_t)__cvta_generic_to_shared(&stage[i % kSlots][threadIdx.x][0]);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s0), "l"(p) : "memory");
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s0 + 16), "l"(p + 2) : "memory");
            asm volatile("cp.async.commit_group;" ::: "memory");
            asm volatile("cp.async.wait_group 7;" ::: "memory");   // the sector staged kSlots - 1 iterations ago has landed
            acc += stage[(i + 1) % kSlots][threadIdx.x][0] ^ stage[(i + 1) % kSlots][threadIdx.x][3];
        } else {
            asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory"); // the slot used two iterations ago is free
            uint64_t *s = &stage[i & 1][threadIdx.x][0];
            s[0] = v; s[1] = v << 1; s[2] = v >> 1; s[3] = v | 1;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            const uint32_t s0 = (uint32_t)__cvta_generic_to_shared(s);
            asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.or.b64 [%0], [%1], 32;" ::"l"(p), "r"(s0) : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
    }
    if (MODE == 3 || MODE == 6) asm volatile("cp.async.wait_group 0;" ::: "memory");
    if (MODE == 4) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    if (acc == 0x1234567u) sink[0] = acc;
}

template <int MODE>
cudaError_t launch_pipe(uint32_t *sink, int iters, long long *cycles, int blocks)
{
    pipe_rate_kernel<MODE><<<blocks, kPipeTPB>>>(sink, iters, 12345u, cycles);
    return cudaGetLastError();
}

template <int MODE>
cudaError_t launch_rand(uint64_t *arr, uint64_t mask, uint32_t per_thread, uint64_t *sink, int blocks)
{
    random_sector_kernel<MODE><<<blocks, kRandTPB>>>(arr, mask, per_thread, sink);
    return cudaGetLastError();
}

} // namespace

extern "C" {

int sbf_ceiling_pipe_modes(void) { return kPipeModes; }
const char *sbf_ceiling_pipe_mode_name(int mode) { return (mode >= 0 && mode < kPipeModes) ? kPipeModeName[mode] : ""; }

int sbf_ceiling_pipe_rate(int mode, int iters, double *g_warp_inst_per_s_per_smsp, double *clock64_mhz)
{
    if (mode < 0 || mode >= kPipeModes || iters < 1 || !g_warp_inst_per_s_per_smsp) return SBF_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return SBF_ERR_CUDA;
    const int blocks = sms * kPipeCTAsPerSM;
    uint32_t *sink = nullptr;
    long long *cyc = nullptr;
    if (cudaMalloc(&sink, 64) != cudaSuccess || cudaMalloc(&cyc, sizeof(long long) * blocks) != cudaSuccess) return SBF_ERR_NOMEM;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaError_t err = cudaSuccess;
    float best_ms = 1e30f;
    double best_cycles = 0;
    long long *h = new long long[blocks];
    for (int rep = 0; rep < 4 && err == cudaSuccess; ++rep) { // first repetition warms up
        cudaEventRecord(e0);
        switch (mode) {
        case 0: err = launch_pipe<0>(sink, iters, cyc, blocks); break;
        case 1: err = launch_pipe<1>(sink, iters, cyc, blocks); break;
        case 2: err = launch_pipe<2>(sink, iters, cyc, blocks); break;
        case 3: err = launch_pipe<3>(sink, iters, cyc, blocks); break;
        case 4: err = launch_pipe<4>(sink, iters, cyc, blocks); break;
        case 5: err = launch_pipe<5>(sink, iters, cyc, blocks); break;
        case 6: err = launch_pipe<6>(sink, iters, cyc, blocks); break;
        case 7: err = launch_pipe<7>(sink, iters, cyc, blocks); break;
        case 8: err = launch_pipe<8>(sink, iters, cyc, blocks); break;
        case 9: err = launch_pipe<9>(sink, iters, cyc, blocks); break;
        case 10: err = launch_pipe<10>(sink, iters, cyc, blocks); break;
        case 11: err = launch_pipe<11>(sink, iters, cyc, blocks); break;
        default: err = launch_pipe<12>(sink, iters, cyc, blocks); break;
        }
        cudaEventRecord(e1);
        if (err == cudaSuccess) err = cudaEventSynchronize(e1);
        if (err != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        cudaMemcpy(h, cyc, sizeof(long long) * blocks, cudaMemcpyDeviceToHost);
        double mean = 0;
        for (int b = 0; b < blocks; ++b) mean += (double)h[b];
        mean /= blocks;
        if (rep > 0 && ms < best_ms) { best_ms = ms; best_cycles = mean; }
    }
    delete[] h;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink); cudaFree(cyc);
    if (err != cudaSuccess) return SBF_ERR_CUDA;
    // all CTAs are resident at once: every SMSP holds kPipeCTAsPerSM * 8 / 4 warps for the whole run
    const double warps_per_smsp = kPipeCTAsPerSM * (kPipeTPB / 32) / 4.0;
    const double inst_per_warp = (double)iters * kPipeUnroll * kPipeChains;
    *g_warp_inst_per_s_per_smsp = warps_per_smsp * inst_per_warp / (best_ms * 1e-3) / 1e9;
    if (clock64_mhz) *clock64_mhz = best_cycles / (best_ms * 1e-3) / 1e6; // rate of the in-kernel cycle counter
    return SBF_OK;
}

int sbf_ceiling_random_sector(int mode, uint64_t array_bytes, double *g_accesses_per_s)
{
    if (mode < 0 || mode > 7 || !g_accesses_per_s || array_bytes < 4096) return SBF_ERR_INVALID_ARG;
    uint64_t sectors = 1;
    while (sectors * 2 * 32 <= array_bytes) sectors *= 2; // power of two
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return SBF_ERR_CUDA;
    uint64_t *arr = nullptr, *sink = nullptr;
    if (cudaMalloc(&arr, sectors * 32) != cudaSuccess || cudaMalloc(&sink, 64) != cudaSuccess) {
        if (arr) cudaFree(arr);
        cudaGetLastError();
        return SBF_ERR_NOMEM;
    }
    cudaMemset(arr, 0, sectors * 32);
    const int blocks = sms * 8;
    const uint32_t per_thread = 1024;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaError_t err = cudaSuccess;
    float best = 1e30f;
    for (int rep = 0; rep < 4 && err == cudaSuccess; ++rep) {
        cudaEventRecord(e0);
        switch (mode) {
        case 0: err = launch_rand<0>(arr, sectors - 1, per_thread, sink, blocks); break;
        case 1: err = launch_rand<1>(arr, sectors - 1, per_thread, sink, blocks); break;
        case 2: err = launch_rand<2>(arr, sectors - 1, per_thread, sink, blocks); break;
        case 3: err = launch_rand<3>(arr, sectors - 1, per_thread, sink, blocks); break;
        case 4: err = launch_rand<4>(arr, sectors - 1, per_thread, sink, blocks); break;
        case 5: err = launch_rand<5>(arr, sectors - 1, per_thread, sink, blocks); break;
        case 6: err = launch_rand<6>(arr, sectors - 1, per_thread, sink, blocks); break;
        default: err = launch_rand<7>(arr, sectors - 1, per_thread, sink, blocks); break;
        }
        cudaEventRecord(e1);
        if (err == cudaSuccess) err = cudaEventSynchronize(e1);
        if (err != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(arr); cudaFree(sink);
    if (err != cudaSuccess) return SBF_ERR_CUDA;
    *g_accesses_per_s = (double)blocks * kRandTPB * per_thread / (best * 1e-3) / 1e9;
    return SBF_OK;
}


// a1 on its own (tests/test_gpu_parity.py::test_pack_kernel_words_and_mask): pack_kernel launched exactly as the
// insert / query calls of the product library launch it, its two outputs copied to the host.
int sbf_bench_pack(const char *d_seq, uint64_t len, int k, uint32_t *h_words, uint16_t *h_mask, uint64_t n_words)
{
    if ((!d_seq && len) || !h_words || !h_mask || k < 1 || k > 64) return SBF_ERR_INVALID_ARG;
    const uint64_t nw = (len + 15) / 16 + sbfk::kPadWords;
    if (n_words > nw) return SBF_ERR_INVALID_ARG;
    uint32_t *packed = nullptr;
    uint16_t *vmask = nullptr;
    if (cudaMalloc(&packed, nw * sizeof(uint32_t)) != cudaSuccess || cudaMalloc(&vmask, nw * sizeof(uint16_t) + 8) != cudaSuccess) {
        cudaFree(packed);
        cudaGetLastError();
        return SBF_ERR_NOMEM;
    }
    const unsigned blocks = (unsigned)(((nw + 1) / 2 + 255) / 256);
    const int aligned = ((reinterpret_cast<uintptr_t>(d_seq) & 15) == 0) ? 1 : 0;
    sbfk::pack_kernel<<<blocks, 256>>>(reinterpret_cast<const uint8_t *>(d_seq), len, packed, vmask, nw, k, aligned, nullptr,
                                       (len + 31) / 32, nullptr);
    cudaError_t err = cudaGetLastError();
    if (err == cudaSuccess) err = cudaMemcpy(h_words, packed, n_words * sizeof(uint32_t), cudaMemcpyDeviceToHost);
    if (err == cudaSuccess) err = cudaMemcpy(h_mask, vmask, n_words * sizeof(uint16_t), cudaMemcpyDeviceToHost);
    cudaFree(packed);
    cudaFree(vmask);
    return err == cudaSuccess ? SBF_OK : SBF_ERR_CUDA;
}

} // extern "C"

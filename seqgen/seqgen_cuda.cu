/*
 * seqgen_cuda.cu — the i.i.d. uniform generator of seqgen.c, on the device.
 *
 * Input generation only (no packing, hashing or filter access).  It exists for the FPR-vs-size experiment
 * (§V-D, Fig. 6: 10^9 random 31-mers), whose 31 GB of query symbols are produced where they are
 * consumed instead of crossing PCIe.  The counter-based generator is restated from seqgen.c so that
 * sg_uniform_device(seed, first, n) holds exactly the bytes seqgen.uniform(seed, first + n)[first:] holds on the host
 * (tests/test_gpu_fpr_size.py checks it), which lets the CPU oracle see any slice of the device-generated stream.
 */
#include <cstdint>
#include <cuda_runtime.h>

namespace {

__device__ __forceinline__ uint64_t mix64(uint64_t z)
{
    z ^= z >> 33; z *= 0xFF51AFD7ED558CCDull;
    z ^= z >> 33; z *= 0xC4CEB9FE1A85EC53ull;
    z ^= z >> 33;
    return z;
}

/* seqgen.c: sg_rnd(seed, stream, index) with stream = ST_BASE = 0 */
__global__ void __launch_bounds__(256) uniform_kernel(uint64_t a, uint8_t *out, uint64_t first, uint64_t n)
{
    // thread t writes the 4 symbols [4t, 4t+4) as one 32-bit store when the output pointer allows it
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t i0 = 4 * t;
    if (i0 >= n) return;
    uint32_t word = 0;
    const int m = (n - i0) < 4 ? (int)(n - i0) : 4;
    for (int j = 0; j < m; ++j) {
        const uint64_t r = mix64(a ^ mix64(first + i0 + j + 0xD1B54A32D192ED03ull));
        word |= (uint32_t)("ACGT"[r >> 62]) << (8 * j);
    }
    if (m == 4 && (reinterpret_cast<uintptr_t>(out) & 3) == 0) {
        reinterpret_cast<uint32_t *>(out)[t] = word;
    } else {
        for (int j = 0; j < m; ++j) out[i0 + j] = (uint8_t)(word >> (8 * j));
    }
}

} // namespace

extern "C" int sg_uniform_device(uint64_t seed, uint8_t *d_out, uint64_t first, uint64_t n, void *stream)
{
    if (n == 0) return 0;
    // host side of sg_rnd: a = mix64(seed + GOLD * (stream + 1)), stream = 0
    uint64_t z = seed + 0x9E3779B97F4A7C15ull;
    z ^= z >> 33; z *= 0xFF51AFD7ED558CCDull;
    z ^= z >> 33; z *= 0xC4CEB9FE1A85EC53ull;
    z ^= z >> 33;
    const uint64_t threads = (n + 3) / 4;
    uniform_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, (cudaStream_t)stream>>>(z, d_out, first, n);
    return (int)cudaGetLastError();
}

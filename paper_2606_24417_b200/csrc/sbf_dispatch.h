// sbf_dispatch.h — table of specialised stream_kernel instances, filled by the sbf_inst_*.cu files.
#pragma once

#include <cstdint>
#include <cuda_runtime.h>

#include "sbf_device.cuh"

namespace sbfk {

typedef cudaError_t (*stream_launch_fn)(const StreamParams &prm, cudaStream_t stream);

struct KernelEntry {
    int k, m, s, H;
    stream_launch_fn insert;     // run flush = four RED.OR.B64
    stream_launch_fn insert_tma; // run flush = one 32-byte TMA reduction (filters much larger than L2)
    stream_launch_fn query;
    stream_launch_fn query_rec; // record mode (one thread per record)
    stream_launch_fn query_long; // the long records record mode listed (one thread per 128-position chunk)
};

template <int K, int M, int S, int H, int MODE>
cudaError_t launch_stream(const StreamParams &prm, cudaStream_t stream)
{
    constexpr bool INSERT = MODE != kModeQuery;
    const uint64_t per = 16ull * (uint64_t)prm.chunk_blocks;
    const uint64_t chunks = (prm.n_pos + per - 1) / per;
    if (chunks == 0) return cudaSuccess;
    uint64_t blocks = (chunks + kStreamTPB - 1) / kStreamTPB;
    if (!INSERT && prm.fallback != nullptr && blocks > 148 * 8) blocks = 148 * 8; // fallback behind record mode: strides
    stream_kernel<K, M, S, H, MODE><<<(unsigned)blocks, kStreamTPB, 0, stream>>>(prm);
    return cudaGetLastError();
}

template <int K, int M, int S, int H>
cudaError_t launch_stream_rec(const StreamParams &prm, cudaStream_t stream)
{
    if (prm.n_rec == 0) return cudaSuccess;
    const uint64_t blocks = (prm.n_rec + kRecTPB - 1) / kRecTPB;
    stream_rec_kernel<K, M, S, H><<<(unsigned)blocks, kRecTPB, 0, stream>>>(prm);
    return cudaGetLastError();
}

template <int K, int M, int S, int H>
cudaError_t launch_stream_long(const StreamParams &prm, cudaStream_t stream)
{
    if (prm.n_rec == 0 || prm.long_groups == nullptr) return cudaSuccess;
    // the group count lives on the device: a fixed grid strides over the list (and exits at once when it is empty)
    stream_long_kernel<K, M, S, H><<<148 * 4, kStreamTPB, 0, stream>>>(prm);
    return cudaGetLastError();
}

#define SBF_ENTRY(K, M, S, H) \
    { K, M, S, H, &sbfk::launch_stream<K, M, S, H, sbfk::kModeInsert>, &sbfk::launch_stream<K, M, S, H, sbfk::kModeInsertTma>, \
      &sbfk::launch_stream<K, M, S, H, sbfk::kModeQuery>, \
      &sbfk::launch_stream_rec<K, M, S, H>, &sbfk::launch_stream_long<K, M, S, H> }

// One table per translation unit (compiled in parallel); each registers itself when the library is loaded.
void register_table(const KernelEntry *entries, int n); // sbf_api.cu
struct TableRegistration {
    TableRegistration(const KernelEntry *entries, int n) { register_table(entries, n); }
};

} // namespace sbfk

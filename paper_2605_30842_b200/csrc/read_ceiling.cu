// read_ceiling.cu — the read-only streaming ceiling SURVEY.md §8(d) asks every GB/s figure to be quoted against:
// what this part gives a kernel that only READS a large buffer once (eq. 5's W).  Two hand-written
// forms of a sum-reduction over the buffer, so that the attention kernel is not its own yardstick:
//   variant 0: 16-byte vector loads (ld.global.nc.L1::no_allocate.v4), 8 independent loads in flight per thread,
//              a grid of 2 x 1024 threads per SM striding the buffer;
//   variant 1: the attention kernel's own transport -- one persistent CTA per SM, one elected lane issuing 8 KiB
//              cp.async.bulk (TMA) copies into a 16-stage shared-memory ring guarded by mbarriers, 128 KiB in
//              flight per SM, four consumer warps summing each stage out of shared memory.
// Every loaded word enters an integer sum that is written out per CTA, so no load can be elided.
#include "../../include/comem_decode_attn.h"
#include "decode_params.cuh"
#include "ptx.cuh"

namespace comem {
namespace {

constexpr int kVecThreads = 1024;
constexpr int kVecUnroll = 8;

__global__ void __launch_bounds__(kVecThreads, 2)
read_vec_kernel(const uint4 *__restrict__ buf, size_t n_vec, unsigned long long *sink)
{
    const size_t stride = (size_t)gridDim.x * kVecThreads;
    size_t i = (size_t)blockIdx.x * kVecThreads + threadIdx.x;
    unsigned acc = 0;
    for (; i + (kVecUnroll - 1) * stride < n_vec; i += kVecUnroll * stride) {
        uint4 v[kVecUnroll];
#pragma unroll
        for (int u = 0; u < kVecUnroll; ++u)
            asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                         : "=r"(v[u].x), "=r"(v[u].y), "=r"(v[u].z), "=r"(v[u].w) : "l"(buf + i + u * stride));
#pragma unroll
        for (int u = 0; u < kVecUnroll; ++u) acc += (v[u].x + v[u].y) + (v[u].z + v[u].w);
    }
    for (; i < n_vec; i += stride) {
        const uint4 v = buf[i];
        acc += (v.x + v.y) + (v.z + v.w);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    __shared__ unsigned s_part[kVecThreads / 32];
    if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = 0;
        for (int w = 0; w < kVecThreads / 32; ++w) t += s_part[w];
        sink[blockIdx.x] = t;
    }
}

constexpr int kTmaStages = 16;
constexpr int kTmaStageBytes = 8192;
constexpr int kTmaConsumerWarps = 4;
constexpr int kTmaThreads = 32 * (kTmaConsumerWarps + 1);
constexpr int kTmaSmem = kTmaStages * kTmaStageBytes + 2 * kTmaStages * 8 + 1024;

__global__ void __launch_bounds__(kTmaThreads, 1)
read_tma_kernel(const uint8_t *__restrict__ buf, size_t n_chunks, unsigned long long *sink)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t ring = (smem_u32(smem_raw) + 127u) & ~127u;
    const uint32_t full0 = ring + kTmaStages * kTmaStageBytes, empty0 = full0 + 8 * kTmaStages;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kTmaStages; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, kTmaConsumerWarps);
        }
        fence_mbar_init();
    }
    __syncthreads();
    // chunk c of the buffer goes to CTA c % grid: neighbouring CTAs read neighbouring 8 KiB pieces
    const size_t first = blockIdx.x, step = gridDim.x;
    if (warp == kTmaConsumerWarps) {
        if (lane == 0) {
            int it = 0;
            for (size_t c = first; c < n_chunks; c += step, ++it) {
                const int s = it % kTmaStages;
                mbar_wait(empty0 + 8 * s, ((uint32_t)(it / kTmaStages) & 1u) ^ 1u);
                mbar_arrive_expect_tx(full0 + 8 * s, kTmaStageBytes);
                bulk_load(ring + s * kTmaStageBytes, buf + c * kTmaStageBytes, kTmaStageBytes, full0 + 8 * s);
            }
        }
        return;
    }
    unsigned acc = 0;
    int it = 0;
    for (size_t c = first; c < n_chunks; c += step, ++it) {
        const int s = it % kTmaStages;
        mbar_wait(full0 + 8 * s, (uint32_t)(it / kTmaStages) & 1u);
        const uint32_t base = ring + s * kTmaStageBytes + (warp * 32 + lane) * 16;
#pragma unroll
        for (int k = 0; k < kTmaStageBytes / (kTmaConsumerWarps * 32 * 16); ++k) {
            const uint4 v = lds128(base + k * kTmaConsumerWarps * 32 * 16);
            acc += (v.x + v.y) + (v.z + v.w);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty0 + 8 * s);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) atomicAdd(sink + blockIdx.x, (unsigned long long)acc);
}

}  // namespace
}  // namespace comem

using namespace comem;

extern "C" int comem_read_ceiling_async(const void *buf, size_t bytes, unsigned long long *sink, int variant,
                                        void *cuda_stream)
{
    if (!buf || !sink || bytes < (size_t)kTmaStageBytes || (reinterpret_cast<uintptr_t>(buf) & 127u) != 0)
        return COMEM_ERR_INVALID_ARG;
    if (variant != 0 && variant != 1) return COMEM_ERR_INVALID_ARG;
    int dev = 0, sms = 0, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
        cudaGetLastError();
        return COMEM_ERR_CUDA;
    }
    if (major != 10) return COMEM_ERR_UNSUPPORTED;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (sms > COMEM_READ_CEILING_SINK_WORDS / 2) sms = COMEM_READ_CEILING_SINK_WORDS / 2;
    if (cudaMemsetAsync(sink, 0, sizeof(unsigned long long) * COMEM_READ_CEILING_SINK_WORDS, stream) != cudaSuccess) {
        cudaGetLastError();
        return COMEM_ERR_CUDA;
    }
    if (variant == 0) {
        read_vec_kernel<<<2 * sms, kVecThreads, 0, stream>>>(static_cast<const uint4 *>(buf), bytes / 16, sink);
    } else {
        static PerDeviceOnce once;
        if (set_max_smem_once(read_tma_kernel, kTmaSmem, once) != cudaSuccess) {
            cudaGetLastError();
            return COMEM_ERR_CUDA;
        }
        read_tma_kernel<<<sms, kTmaThreads, kTmaSmem, stream>>>(static_cast<const uint8_t *>(buf), bytes / kTmaStageBytes, sink);
    }
    if (cudaGetLastError() != cudaSuccess) return COMEM_ERR_CUDA;
    return COMEM_OK;
}

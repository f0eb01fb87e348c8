// Read-only ceiling probe (SURVEY.md 8(d) "How to measure": "a trivial read-only sum kernel over >= 16 GB as the achievable
// ceiling"): the demodulation kernels read every sample once and write almost nothing (the paper's point that QLD needs two n^2
// arrays beside the frames), so the bandwidth that bounds them is what the GPU sustains on READS alone -- higher than
// the read+write copy figure the roofline peak is measured with.  This kernel is that measurement: every byte of a buffer is
// loaded once (16-byte loads that bypass L1, eight in flight per thread) and folded into one word per CTA; nothing else happens.
// It is a measuring stick for bench.py, not a step of the path.
#include <cuda_runtime.h>
#include <stdint.h>

#include "qld_internal.h"

namespace {

constexpr int PROBE_THREADS = 512;
constexpr int PROBE_UNROLL = 8;

__device__ __forceinline__ uint4 ld_stream16(const uint4 *p)
{
    uint4 v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::256B.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}

__global__ void __launch_bounds__(PROBE_THREADS) k_probe_read(const uint4 *buf, int64_t n16, uint32_t *out)
{
    uint32_t acc = 0;
    const int64_t stride = (int64_t)gridDim.x * PROBE_THREADS;
    int64_t i = (int64_t)blockIdx.x * PROBE_THREADS + threadIdx.x;
    for (; i + (PROBE_UNROLL - 1) * stride < n16; i += PROBE_UNROLL * stride) {
        uint4 v[PROBE_UNROLL];
#pragma unroll
        for (int u = 0; u < PROBE_UNROLL; ++u) v[u] = ld_stream16(buf + i + u * stride);
#pragma unroll
        for (int u = 0; u < PROBE_UNROLL; ++u) acc += v[u].x ^ v[u].y ^ v[u].z ^ v[u].w;
    }
    for (; i < n16; i += stride) {
        const uint4 v = ld_stream16(buf + i);
        acc += v.x ^ v.y ^ v.z ^ v.w;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    __shared__ uint32_t part[PROBE_THREADS / 32];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int w = 0; w < PROBE_THREADS / 32; ++w) t += part[w];
        out[blockIdx.x] = t;
    }
}

}  // namespace

extern "C" int qld_probe_read(const void *buf_device, int64_t bytes, uint32_t *out_device, void *stream)
{
    if (!buf_device || !out_device || bytes < 16 || (reinterpret_cast<uintptr_t>(buf_device) & 15) != 0) return QLD_E_INVAL;
    const int grid = qld_sm_count() * 4;                       // 4 x 512 threads per SM: the SM's full complement of warps
    if (grid > QLD_PROBE_OUT_WORDS) return QLD_E_UNSUPPORTED;
    k_probe_read<<<grid, PROBE_THREADS, 0, static_cast<cudaStream_t>(stream)>>>(static_cast<const uint4 *>(buf_device), bytes / 16, out_device);
    return cudaGetLastError() == cudaSuccess ? QLD_OK : QLD_E_CUDA;
}

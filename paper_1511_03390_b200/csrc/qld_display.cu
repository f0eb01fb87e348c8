// Headless stand-in for the paper's display step (the 32-bit processed image "is displayed on the computer
// monitor", second half): the range of a float32 map and its linear mapping to 8 bits.  Two launches:
// a grid-stride min/max reduction (ordered-integer atomics, so the result does not depend on the order of arrival) and
// the mapping u8 = rint(255 * (x - lo) / (hi - lo)), clamped; a flat map becomes all zeros.  No graphics API is involved:
// the 8-bit image lands in device memory.
#include <cuda_runtime.h>
#include <stdint.h>

#include "qld_internal.h"

namespace {

// order-preserving map float -> uint32 (finite values and infinities; NaNs are skipped by the caller)
__device__ __forceinline__ uint32_t f2ord(float f)
{
    const uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ord2f(uint32_t o)
{
    return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o);
}

__global__ void k_range_init(uint32_t *mm)
{
    mm[0] = 0xffffffffu;   // min
    mm[1] = 0u;            // max
}

__global__ void __launch_bounds__(256) k_range(const float *x, int64_t n, uint32_t *mm)
{
    uint32_t lo = 0xffffffffu, hi = 0u;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float v = x[i];
        if (v == v) {
            const uint32_t o = f2ord(v);
            lo = o < lo ? o : lo;
            hi = o > hi ? o : hi;
        }
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        const uint32_t l2 = __shfl_xor_sync(0xffffffffu, lo, s), h2 = __shfl_xor_sync(0xffffffffu, hi, s);
        lo = l2 < lo ? l2 : lo;
        hi = h2 > hi ? h2 : hi;
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMin(&mm[0], lo);
        atomicMax(&mm[1], hi);
    }
}

__global__ void __launch_bounds__(256) k_to_u8(const float *x, int64_t n, const uint32_t *mm, float *range_out, uint8_t *out)
{
    const float lo = ord2f(mm[0]), hi = ord2f(mm[1]);
    if (range_out && blockIdx.x == 0 && threadIdx.x == 0) { range_out[0] = lo; range_out[1] = hi; }
    const double span = (double)hi - (double)lo;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float v = x[i];
        double t = span > 0.0 && v == v ? rint(255.0 * ((double)v - (double)lo) / span) : 0.0;
        t = t < 0.0 ? 0.0 : (t > 255.0 ? 255.0 : t);
        out[i] = (uint8_t)t;
    }
}

}  // namespace

extern "C" int qld_display_map(const float *map_device, int64_t n, uint8_t *out_device, float *range_device, void *scratch_device, void *stream)
{
    if (!map_device || !out_device || !scratch_device || n < 1) return QLD_E_INVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    uint32_t *mm = static_cast<uint32_t *>(scratch_device);
    const int cap = qld_sm_count() * 8;
    const int blocks = (int)((n + 255) / 256 < cap ? (n + 255) / 256 : cap);
    k_range_init<<<1, 1, 0, st>>>(mm);
    k_range<<<blocks, 256, 0, st>>>(map_device, n, mm);
    k_to_u8<<<blocks, 256, 0, st>>>(map_device, n, mm, range_device, out_device);
    return cudaGetLastError() == cudaSuccess ? QLD_OK : QLD_E_CUDA;
}

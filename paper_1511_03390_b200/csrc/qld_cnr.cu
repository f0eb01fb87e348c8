// Contrast-to-noise ratio of a processed image (Eq. (1), Fig. 6) -- the step after the hot path
// (SURVEY.md 8(f1)): mean over the m x m source square, mean and rms deviation over the m-pixel wide square slice
// around it (8 m^2 pixels).  One block; the regions are a few thousand pixels, so this is a latency-sized reduction:
// two passes over the slice in fp64 (mean first, then the deviations from it, as Eq. (1) is written).
#include <cuda_runtime.h>
#include <stdint.h>

#include "qld.h"

namespace {

constexpr int CNR_THREADS = 256;

__device__ double block_sum(double v, double *scratch)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();                                     // scratch may still be read from the previous call
    if (lane == 0) scratch[warp] = v;
    __syncthreads();
    double t = 0.0;
    for (int i = 0; i < CNR_THREADS / 32; ++i) t += scratch[i];   // same order in every thread: one value for all
    return t;
}

__global__ void __launch_bounds__(CNR_THREADS) k_cnr(const float *img, int W, int y0, int x0, int m, double *out)
{
    __shared__ double scratch[CNR_THREADS / 32];
    const int side = 3 * m, n_big = side * side;
    double s_src = 0.0, s_ring = 0.0;
    for (int i = threadIdx.x; i < n_big; i += CNR_THREADS) {
        const int dy = i / side, dx = i % side;
        const double v = (double)img[(int64_t)(y0 - m + dy) * W + (x0 - m + dx)];
        const bool in_src = dy >= m && dy < 2 * m && dx >= m && dx < 2 * m;
        if (in_src) s_src += v; else s_ring += v;
    }
    const double mean_s = block_sum(s_src, scratch) / (double)(m * m);
    const double mean_r = block_sum(s_ring, scratch) / (double)(8 * m * m);
    double dev = 0.0;
    for (int i = threadIdx.x; i < n_big; i += CNR_THREADS) {
        const int dy = i / side, dx = i % side;
        const bool in_src = dy >= m && dy < 2 * m && dx >= m && dx < 2 * m;
        if (!in_src) {
            const double d = (double)img[(int64_t)(y0 - m + dy) * W + (x0 - m + dx)] - mean_r;
            dev += d * d;
        }
    }
    const double rms = sqrt(block_sum(dev, scratch) / (double)(8 * m * m));
    if (threadIdx.x == 0) {
        out[0] = (mean_s - mean_r) / rms;                // IEEE: inf / nan when the slice is flat
        out[1] = mean_s;
        out[2] = mean_r;
        out[3] = rms;
    }
}

}  // namespace

extern "C" int qld_cnr(const float *map_device, int32_t H, int32_t W, int32_t y0, int32_t x0, int32_t m, double *out_device, void *stream)
{
    if (!map_device || !out_device || H < 1 || W < 1 || m < 1) return QLD_E_INVAL;
    if (m > 10000 || y0 - m < 0 || x0 - m < 0 || (int64_t)y0 + 2 * (int64_t)m > H || (int64_t)x0 + 2 * (int64_t)m > W) return QLD_E_INVAL;
    k_cnr<<<1, CNR_THREADS, 0, static_cast<cudaStream_t>(stream)>>>(map_device, W, y0, x0, m, out_device);
    return cudaGetLastError() == cudaSuccess ? QLD_OK : QLD_E_CUDA;
}

// Unknown-frequency search: the paper's Fourier decomposition "is essentially a series of QLDs being
// performed at different frequencies", and the FFT image is |F(j,k,omega_q)|^2 at the bin of interest
// (PAPER.md:99).  When the modulation frequency is not known, every bin q_lo..q_hi of the N-frame window (nu = q/N) is
// demodulated -- eight bins per pass over the stack, on the tensor-core path where it applies -- and each pixel keeps
// the bin with the largest amplitude R_q = |F_q|.  Built on the public C ABI only (qld_create .. qld_destroy) plus one
// small kernel that folds a pass's amplitude maps into the running maximum.
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include "qld.h"

namespace {

__global__ void k_peak_update(const float *amp, int K, int64_t HW, int q0, int first, float *best, int32_t *bin)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= HW) return;
    float b = first ? -1.0f : best[p];
    int q = first ? q0 : bin[p];
    for (int k = 0; k < K; ++k) {
        const float a = amp[(int64_t)k * HW + p];
        if (a > b) { b = a; q = q0 + k; }               // strict: the lowest bin wins a tie
    }
    best[p] = b;
    bin[p] = q;
}

}  // namespace

extern "C" int qld_dominant_bin(const void *frames_device, int32_t dtype, int32_t H, int32_t W, int32_t N, int32_t q_lo, int32_t q_hi,
                                float *amp_max_device, int32_t *bin_device, void *stream)
{
    if (!frames_device || !amp_max_device || !bin_device || H < 1 || W < 1 || N < 3) return QLD_E_INVAL;
    if (q_lo < 1 || q_hi < q_lo || 2 * (int64_t)q_hi >= N) return QLD_E_INVAL;       // 0 < q/N < 1/2 (reading G18)
    cudaStream_t st = stream ? static_cast<cudaStream_t>(stream) : cudaStreamLegacy;
    const int64_t HW = (int64_t)H * W;
    int first = 1;
    for (int q0 = q_lo; q0 <= q_hi; q0 += 8) {
        const int K = q_hi - q0 + 1 < 8 ? q_hi - q0 + 1 : 8;
        qld_ref refs[8];
        memset(refs, 0, sizeof refs);
        for (int k = 0; k < K; ++k) { refs[k].num = q0 + k; refs[k].den = N; }
        qld_config cfg;
        memset(&cfg, 0, sizeof cfg);
        cfg.H = H; cfg.W = W; cfg.dtype = dtype; cfg.N = N; cfg.K = K; cfg.refs = refs;
        cfg.ring_frames = -1; cfg.maps = QLD_MAP_AMP; cfg.compute_stream = st;
        qld_ctx *ctx = nullptr;
        cfg.accum = QLD_ACC_FIXED;                      // exact sums, one precision for every pass ...
        int rc = qld_create(&cfg, &ctx);
        if (rc == QLD_E_UNSUPPORTED) {                  // ... unless the frame does not fit the tensor-core path
            cfg.accum = QLD_ACC_FP32;
            rc = qld_create(&cfg, &ctx);
        }
        if (rc != QLD_OK) return rc;
        rc = qld_attach_frames_device(ctx, frames_device);
        if (rc == QLD_OK) rc = qld_demod(ctx, QLD_WHOLE, 0);
        const float *amp = nullptr;
        if (rc == QLD_OK) rc = qld_get_maps(ctx, 0, nullptr, nullptr, &amp, nullptr);
        if (rc == QLD_OK) {
            k_peak_update<<<(unsigned)((HW + 255) / 256), 256, 0, st>>>(amp, K, HW, q0, first, amp_max_device, bin_device);
            if (cudaGetLastError() != cudaSuccess) rc = QLD_E_CUDA;
        }
        qld_destroy(ctx);                               // waits for the pass (the context owns the maps)
        if (rc != QLD_OK) return rc;
        first = 0;
    }
    return QLD_OK;
}

// Device twin of paper_1511_03390_b200/synth.py: fills synthetic frames straight into device memory so the
// large benchmark stacks (GBs) need no host generation.  Inputs only: none of the QLD arithmetic is here.
// Every floating-point step is a single correctly-rounded IEEE operation (__dmul_rn, __dadd_rn, __dsqrt_rn,
// rint), in the order synth.py states, so the bytes are identical to the numpy generator.
#include "qld_internal.h"

namespace {

__device__ __forceinline__ uint64_t mix64(uint64_t x)
{
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}
__device__ __forceinline__ int field_sum(uint64_t h)
{
    return (int)(h & 0xFFFF) + (int)((h >> 16) & 0xFFFF) + (int)((h >> 32) & 0xFFFF) + (int)(h >> 48);
}

__global__ void k_synth_fill(const qld_synth_scene sc, int64_t s_first, int n_frames, void *out)
{
    const uint64_t GOLDEN = 0x9E3779B97F4A7C15ull;
    const int64_t HW = (int64_t)sc.H * sc.W;
    const int64_t total = HW * n_frames;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int64_t f = idx / HW, p = idx - f * HW;
        const int64_t s = s_first + f;
        const uint64_t c = (uint64_t)s * (uint64_t)HW + (uint64_t)p;
        const uint64_t ha = mix64(sc.key + (c * 2ull) * GOLDEN);
        const uint64_t hb = mix64(sc.key + (c * 2ull + 1ull) * GOLDEN);
        const double z = __dmul_rn((double)(field_sum(ha) + field_sum(hb) - 262140), 1.8688123650118534e-05);
        double lam = (double)sc.base[p];
        for (int j = 0; j < sc.n_terms; ++j)
            lam = __dadd_rn(lam, __dmul_rn((double)sc.weights[(int64_t)j * HW + p], sc.mods[(int64_t)j * sc.mod_stride + s]));
        if (sc.has_disk) {
            const int64_t px = p % sc.W, py = p / sc.W;
            int64_t dx = (px - sc.disk_x0 - s) % sc.W;
            if (dx < 0) dx += sc.W;
            if (dx >= sc.W - dx) dx -= sc.W;
            const int64_t dy = py - sc.disk_cy;
            if (dx * dx + dy * dy <= (int64_t)sc.disk_radius * sc.disk_radius)
                lam = __dadd_rn(lam, __dmul_rn(sc.disk_amp, sc.disk_mod[s]));
        }
        const double var = __dadd_rn(sc.noise_a, __dmul_rn(sc.noise_b, lam));
        double x = rint(__dadd_rn(lam, __dmul_rn(__dsqrt_rn(var), z)));
        x = fmin(fmax(x, 0.0), (double)sc.maxval);
        if (sc.dtype == QLD_U8) static_cast<uint8_t *>(out)[idx] = (uint8_t)x;
        else static_cast<uint16_t *>(out)[idx] = (uint16_t)x;
    }
}

}  // namespace

extern "C" int qld_synth_fill(const qld_synth_scene *scene, int64_t s_first, int n_frames, void *out_device, void *stream)
{
    if (!scene || !out_device || n_frames < 1 || scene->H < 1 || scene->W < 1 || scene->n_terms < 0 || scene->n_terms > 8) return QLD_E_INVAL;
    const int64_t total = (int64_t)scene->H * scene->W * n_frames;
    const int64_t blocks = (total + 255) / 256;
    const int64_t cap = (int64_t)qld_sm_count() * 32;
    const unsigned grid = (unsigned)(blocks < cap ? blocks : cap);
    k_synth_fill<<<grid, 256, 0, static_cast<cudaStream_t>(stream)>>>(*scene, s_first, n_frames, out_device);
    return cudaGetLastError() == cudaSuccess ? QLD_OK : QLD_E_CUDA;
}

// Demodulation kernels of the QLD hot path (SURVEY.md section 8(a) rows A3, A3', A4, A5, A6) for sm_100a.
//
// What they compute (readings G1-G6):
//   row_r(p) = sum_s x_s(p) * w_r(s)      over the frames of one window, for ROWS weight rows at once,
// where the weight rows are either (sin theta_{k,s}, cos theta_{k,s}) pairs in fp32 (2K rows) or integer
// phase-bin indicators in {0,+1,-1}; then, fused, I_k, Q_k, amplitude sqrt(I^2+Q^2) and phase atan2(Q, I).
// The paper's two "intermediate frames" never exist in memory: products live in registers.
//
// Design: HBM-bound streaming reduction.  Each thread owns V adjacent pixels (one 16-byte load per frame),
// the CTA's warps split the time axis (threadIdx.y), every sample is read exactly once, the 2K (or bin)
// accumulators stay in registers, and the time slices are combined through shared memory at the end.
#include "qld_device.cuh"

using namespace qld_dev;

namespace {

// ---------------------------------------------------------------------------------------------------
// A3 / A3' / A6: whole-window demodulation.  blockDim = (BX, TY): x = pixel vectors, y = time slices.
// shared memory: RED red[ROWS][V][BX] + float ped[V][BX].
// ---------------------------------------------------------------------------------------------------
template <typename T, typename ACC, int ROWS, int V>
__global__ void __launch_bounds__(256) k_demod_whole(const DemodParams p)
{
    using PX = Pix<T, V>;
    constexpr bool IS_INT = std::is_same<ACC, int>::value;
    using RED = typename std::conditional<IS_INT, int, double>::type;
    constexpr int U = (ROWS * V >= 64) ? 2 : 4;   // frames in flight per thread per iteration

    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int BX = blockDim.x, TY = blockDim.y, tx = threadIdx.x, ty = threadIdx.y;
    RED *red = reinterpret_cast<RED *>(smem_raw);
    float *pedsm = reinterpret_cast<float *>(smem_raw + (size_t)ROWS * V * BX * sizeof(RED));

    const int64_t pix0 = ((int64_t)blockIdx.x * BX + tx) * V;
    const bool active = pix0 < p.HW;
    const unsigned char *base = static_cast<const unsigned char *>(p.frames) + pix0 * (int64_t)sizeof(T);
    const ACC *wtab = static_cast<const ACC *>(p.wtab);

    const uint32_t bsw = p.big_endian ? 0x11u : 0u;
    ACC acc[ROWS][V];
#pragma unroll
    for (int r = 0; r < ROWS; ++r)
#pragma unroll
        for (int v = 0; v < V; ++v) acc[r][v] = 0;
    float pedm[V];
#pragma unroll
    for (int v = 0; v < V; ++v) pedm[v] = 8388608.0f;

    if (active) {
        if constexpr (!IS_INT) {
            // pedestal = the pixel's first sample in the window (exact integer), DESIGN.md "Precision"
            uint32_t w0[PX::NW];
            PX::load(base + (int64_t)p.slot0 * p.frame_stride, w0);
#pragma unroll
            for (int v = 0; v < V; ++v) pedm[v] = PX::getf_biased(w0, v, bsw);
            if (ty == 0) {
#pragma unroll
                for (int v = 0; v < V; ++v) pedsm[v * BX + tx] = pedm[v] - 8388608.0f;
            }
        }
        const int len = (p.n + TY - 1) / TY;
        int f = ty * len;
        const int f1 = min(p.n, f + len);
        int slot = p.slot0 + f;
        if (slot >= p.cap) slot -= p.cap;
        int we = p.w0 + f;
        if (we >= p.cap_w) we -= p.cap_w;
        for (; f + U <= f1; f += U) {
            uint32_t w[U][PX::NW];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                int s = slot + u;
                if (s >= p.cap) s -= p.cap;
                PX::load(base + (int64_t)s * p.frame_stride, w[u]);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                int e = we + u;
                if (e >= p.cap_w) e -= p.cap_w;
                ACC wt[ROWS];
                load_weights<ACC, ROWS>(wtab + (int64_t)e * ROWS, wt);
                accumulate<T, ACC, ROWS, V>(w[u], wt, pedm, acc, bsw);
            }
            slot += U;
            if (slot >= p.cap) slot -= p.cap;
            we += U;
            if (we >= p.cap_w) we -= p.cap_w;
        }
        for (; f < f1; ++f) {
            uint32_t w[PX::NW];
            PX::load(base + (int64_t)slot * p.frame_stride, w);
            ACC wt[ROWS];
            load_weights<ACC, ROWS>(wtab + (int64_t)we * ROWS, wt);
            accumulate<T, ACC, ROWS, V>(w, wt, pedm, acc, bsw);
            if (++slot >= p.cap) slot -= p.cap;
            if (++we >= p.cap_w) we -= p.cap_w;
        }
    }

    // combine the TY time slices: slice 0 stores, the others add in turn (fp64 / int32)
    for (int yy = 0; yy < TY; ++yy) {
        if (ty == yy && active) {
#pragma unroll
            for (int r = 0; r < ROWS; ++r)
#pragma unroll
                for (int v = 0; v < V; ++v) {
                    RED *cell = &red[(r * V + v) * BX + tx];
                    if (yy == 0) *cell = (RED)acc[r][v];
                    else *cell += (RED)acc[r][v];
                }
        }
        __syncthreads();
    }
    if (!active) return;

    // A4 epilogue: the slices share the V pixels of their column
    for (int v = ty; v < V; v += TY) {
        const int64_t pixel = pix0 + v;
        double val[ROWS];
        if constexpr (IS_INT) {
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                int b = red[(r * V + v) * BX + tx];
                val[r] = (double)b;
                if (p.acc_out) static_cast<int *>(p.acc_out)[(int64_t)r * p.HW + pixel] = b;
            }
        } else {
            const double ped = (double)pedsm[v * BX + tx];
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                double a = red[(r * V + v) * BX + tx];
                if (p.acc_out) static_cast<double *>(p.acc_out)[(int64_t)r * p.HW + pixel] = a;
                const double wsum = p.cum[(int64_t)p.cum_hi * ROWS + r] - p.cum[(int64_t)p.cum_lo * ROWS + r];
                val[r] = a + ped * wsum;     // sum x w = sum (x - ped) w + ped * sum w
            }
            if (p.ped_out) p.ped_out[pixel] = (float)ped;
        }
        finalise_pixel<ROWS>(p.fin, val, pixel, p.HW);
    }
}

// ---------------------------------------------------------------------------------------------------
// A5: sliding-window update.  acc += sum over the hop new frames - sum over the hop expired frames, each
// partial computed from zero in frame order, accumulators fp64 (FP32 mode) or int32 (bins, exact).  With a
// constant hop the fp32 partial a batch adds here is the one this kernel later removes, but the seed comes from
// another kernel with another time slicing, and k_demod_stream folds -expired and +new into one fp32 sum: FP32
// ring sums therefore drift (a random walk of rounding errors) and qld_demod resynchronises them from the ring
// every cfg.resync_hops hops (default: every 16 windows' worth).  One thread = V pixels.
// ---------------------------------------------------------------------------------------------------
template <typename T, typename ACC, int ROWS, int V>
__device__ __forceinline__ void hop_partial(const unsigned char *base, int64_t stride, int cap, int slot, const ACC *wtab, int cap_w,
                                            int we, int hop, const float (&pedm)[V], ACC (&acc)[ROWS][V], uint32_t bsw)
{
    using PX = Pix<T, V>;
    constexpr int U = (ROWS * V >= 64) ? 2 : 4;
    int f = 0;
    for (; f + U <= hop; f += U) {
        uint32_t w[U][PX::NW];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            int s = slot + u;
            if (s >= cap) s -= cap;
            PX::load(base + (int64_t)s * stride, w[u]);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            int e = we + u;
            if (e >= cap_w) e -= cap_w;
            ACC wt[ROWS];
            load_weights<ACC, ROWS>(wtab + (int64_t)e * ROWS, wt);
            accumulate<T, ACC, ROWS, V>(w[u], wt, pedm, acc, bsw);
        }
        slot += U;
        if (slot >= cap) slot -= cap;
        we += U;
        if (we >= cap_w) we -= cap_w;
    }
    for (; f < hop; ++f) {
        uint32_t w[PX::NW];
        PX::load(base + (int64_t)slot * stride, w);
        ACC wt[ROWS];
        load_weights<ACC, ROWS>(wtab + (int64_t)we * ROWS, wt);
        accumulate<T, ACC, ROWS, V>(w, wt, pedm, acc, bsw);
        if (++slot >= cap) slot -= cap;
        if (++we >= cap_w) we -= cap_w;
    }
}

template <typename T, typename ACC, int ROWS, int V>
__global__ void __launch_bounds__(128) k_demod_slide(const SlideParams p)
{
    constexpr bool IS_INT = std::is_same<ACC, int>::value;
    const int64_t pix0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * V;
    if (pix0 >= p.HW) return;
    const unsigned char *base = static_cast<const unsigned char *>(p.frames) + pix0 * (int64_t)sizeof(T);
    const ACC *wtab = static_cast<const ACC *>(p.wtab);

    float pedm[V];
#pragma unroll
    for (int v = 0; v < V; ++v) pedm[v] = 8388608.0f + (IS_INT ? 0.0f : p.ped[pix0 + v]);

    ACC a_new[ROWS][V], a_old[ROWS][V];
#pragma unroll
    for (int r = 0; r < ROWS; ++r)
#pragma unroll
        for (int v = 0; v < V; ++v) {
            a_new[r][v] = 0;
            a_old[r][v] = 0;
        }
    hop_partial<T, ACC, ROWS, V>(base, p.frame_stride, p.cap, p.new_slot0, wtab, p.cap_w, p.new_w0, p.hop, pedm, a_new, p.big_endian ? 0x11u : 0u);
    hop_partial<T, ACC, ROWS, V>(base, p.frame_stride, p.cap, p.old_slot0, wtab, p.cap_w, p.old_w0, p.hop, pedm, a_old, p.big_endian ? 0x11u : 0u);

#pragma unroll
    for (int v = 0; v < V; ++v) {
        const int64_t pixel = pix0 + v;
        double val[ROWS];
        if constexpr (IS_INT) {
            int *acc = static_cast<int *>(p.acc);
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                int b = acc[(int64_t)r * p.HW + pixel] + (a_new[r][v] - a_old[r][v]);
                acc[(int64_t)r * p.HW + pixel] = b;
                val[r] = (double)b;
            }
        } else {
            double *acc = static_cast<double *>(p.acc);
            const double ped = (double)(pedm[v] - 8388608.0f);
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                double a = acc[(int64_t)r * p.HW + pixel] + ((double)a_new[r][v] - (double)a_old[r][v]);
                acc[(int64_t)r * p.HW + pixel] = a;
                const double wsum = p.cum[(int64_t)p.cum_hi * ROWS + r] - p.cum[(int64_t)p.cum_lo * ROWS + r];
                val[r] = a + ped * wsum;
            }
        }
        finalise_pixel<ROWS>(p.fin, val, pixel, p.HW);
    }
}

template <typename T, typename ACC, int ROWS>
cudaError_t launch_whole_t(const DemodParams &p, bool vec, cudaStream_t st)
{
    constexpr int V = pick_v(sizeof(T), ROWS);
    constexpr bool IS_INT = std::is_same<ACC, int>::value;
    const int BX = 32;
    const int TY = p.n >= 64 ? 8 : (p.n >= 8 ? p.n / 8 : 1);
    dim3 block(BX, TY);
    const int v = vec ? V : 1;
    const size_t smem = (size_t)ROWS * v * BX * (IS_INT ? sizeof(int) : sizeof(double)) + (size_t)v * BX * sizeof(float);
    const int64_t nvec = (p.HW + v - 1) / v;
    dim3 grid((unsigned)((nvec + BX - 1) / BX));
    if (vec) k_demod_whole<T, ACC, ROWS, V><<<grid, block, smem, st>>>(p);
    else k_demod_whole<T, ACC, ROWS, 1><<<grid, block, smem, st>>>(p);
    return cudaGetLastError();
}

template <typename T, typename ACC, int ROWS>
cudaError_t launch_slide_t(const SlideParams &p, bool vec, cudaStream_t st)
{
    constexpr int V = pick_v(sizeof(T), ROWS) > 1 ? pick_v(sizeof(T), 2 * ROWS) : 1;   // two partials live at once
    const int v = vec ? V : 1;
    const int64_t nvec = (p.HW + v - 1) / v;
    dim3 block(128), grid((unsigned)((nvec + 127) / 128));
    if (vec) k_demod_slide<T, ACC, ROWS, V><<<grid, block, 0, st>>>(p);
    else k_demod_slide<T, ACC, ROWS, 1><<<grid, block, 0, st>>>(p);
    return cudaGetLastError();
}

template <typename T, typename ACC>
cudaError_t launch_whole_r(int rows, const DemodParams &p, bool vec, cudaStream_t st)
{
    switch (rows) {
    case 2: return launch_whole_t<T, ACC, 2>(p, vec, st);
    case 3: return launch_whole_t<T, ACC, 3>(p, vec, st);
    case 4: return launch_whole_t<T, ACC, 4>(p, vec, st);
    case 8: return launch_whole_t<T, ACC, 8>(p, vec, st);
    case 16: return launch_whole_t<T, ACC, 16>(p, vec, st);
    default: return cudaErrorInvalidValue;
    }
}
template <typename T, typename ACC>
cudaError_t launch_slide_r(int rows, const SlideParams &p, bool vec, cudaStream_t st)
{
    switch (rows) {
    case 2: return launch_slide_t<T, ACC, 2>(p, vec, st);
    case 3: return launch_slide_t<T, ACC, 3>(p, vec, st);
    case 4: return launch_slide_t<T, ACC, 4>(p, vec, st);
    case 8: return launch_slide_t<T, ACC, 8>(p, vec, st);
    case 16: return launch_slide_t<T, ACC, 16>(p, vec, st);
    default: return cudaErrorInvalidValue;
    }
}

bool can_vectorise(int bytes, int v, int64_t HW, const void *frames, int64_t stride)
{
    const int64_t vb = (int64_t)v * bytes;
    return v > 1 && HW % v == 0 && stride % vb == 0 && (reinterpret_cast<uintptr_t>(frames) % vb) == 0;
}

}  // namespace

int qld_pixels_per_thread(int dtype, int rows, int64_t HW, const void *frames, int64_t frame_stride)
{
    const int bytes = dtype == QLD_U8 ? 1 : 2;
    const int v = pick_v(bytes, rows);
    return can_vectorise(bytes, v, HW, frames, frame_stride) ? v : 1;
}

cudaError_t qld_launch_demod_whole(int dtype, int is_int, int rows, const DemodParams &p, cudaStream_t st)
{
    const int bytes = dtype == QLD_U8 ? 1 : 2;
    const bool vec = can_vectorise(bytes, pick_v(bytes, rows), p.HW, p.frames, p.frame_stride);
    if (dtype == QLD_U8) return is_int ? launch_whole_r<uint8_t, int>(rows, p, vec, st) : launch_whole_r<uint8_t, float>(rows, p, vec, st);
    return is_int ? launch_whole_r<uint16_t, int>(rows, p, vec, st) : launch_whole_r<uint16_t, float>(rows, p, vec, st);
}

cudaError_t qld_launch_demod_slide(int dtype, int is_int, int rows, const SlideParams &p, cudaStream_t st)
{
    const int bytes = dtype == QLD_U8 ? 1 : 2;
    const int v = pick_v(bytes, rows) > 1 ? pick_v(bytes, 2 * rows) : 1;
    const bool vec = can_vectorise(bytes, v, p.HW, p.frames, p.frame_stride);
    if (dtype == QLD_U8) return is_int ? launch_slide_r<uint8_t, int>(rows, p, vec, st) : launch_slide_r<uint8_t, float>(rows, p, vec, st);
    return is_int ? launch_slide_r<uint16_t, int>(rows, p, vec, st) : launch_slide_r<uint16_t, float>(rows, p, vec, st);
}

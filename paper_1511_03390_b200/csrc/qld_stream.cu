// TMA-fed whole-window demodulation on the CUDA cores (SURVEY.md 8(a) rows A3, A3', A4, A6 for small K).
//
// Same arithmetic as k_demod_whole: row_r(p) = sum_s x_s(p) * w_r(s), then I, Q,
// amplitude, phase.  What differs is how the bytes travel.  Measured on B200 (read-only probe over the cfg2 stack):
// HBM delivers 7.0-7.2 TB/s when every frame contributes >= 2 KB of contiguous bytes to a request stream and only
// about 6.0 TB/s for isolated 128..512-byte pieces, and a register-staged kernel cannot keep enough bytes in flight
// per SM (80 registers/thread -> 48 KB) to cover the DRAM latency at that rate.  So here one producer thread per SM
// asks the TMA for boxes of {SEG contiguous bytes} x {KC frames} into a ring of shared-memory stages (about 190 KB in
// flight per SM, independent of registers), and eight consumer warps do nothing but LDS -> unpack -> FMA.
//
// One persistent CTA per SM: warp 0 = producer (TMA + the stage's weight rows), warps 1..8 = consumers.  A tile is
// SEG bytes of every frame of the window; tiles are claimed from a global counter.  Inside a tile, consumer warp w
// owns column group (w % CG) -- 32 lanes x V pixels -- and time slice (w / CG): it takes every TS-th frame of each
// stage.  Slices are combined through shared memory at the end of the tile (fp64 / int32), then the A4 epilogue.
#include <stdio.h>
#include <stdlib.h>

#include "qld_device.cuh"
#include "qld_ptx.cuh"
#include "qld_stream.h"

using namespace qld_dev;
using namespace qld_ptx;

namespace {

constexpr int NW = 8;                 // consumer warps
constexpr int TQ = 16;                // tile-id queue entries (producer runs at most `stages` <= 12 tiles ahead)

struct StreamSmem {
    int data_stage, w_stage, off_w, off_red, off_bar, total;
    __host__ __device__ StreamSmem(int seg, int kc, int stages, int rows, int red_bytes)
    {
        data_stage = seg * kc;
        w_stage = kc * rows * 4;
        off_w = stages * data_stage;
        off_red = off_w + stages * w_stage;
        off_bar = off_red + red_bytes;
        total = off_bar + 2 * stages * 8 + TQ * 4 + 16;
    }
};

template <typename T, typename ACC, int ROWS, int V>
__global__ void __launch_bounds__(32 * (NW + 1), 1)
k_demod_stream(const __grid_constant__ CUtensorMap tmap, const DemodParams p, const StreamShape sh, unsigned int *tile_counter)
{
    using PX = Pix<T, V>;
    constexpr bool IS_INT = std::is_same<ACC, int>::value;
    using RED = typename std::conditional<IS_INT, int, double>::type;
    constexpr int VB = V * (int)sizeof(T);                 // bytes per thread per frame

    const int SEG = sh.seg, KC = sh.kc, STAGES = sh.stages;
    const int CG = SEG / (32 * VB), TS = NW / CG;          // column groups, time slices
    const StreamSmem SM(SEG, KC, STAGES, ROWS, TS > 1 ? ROWS * V * CG * 32 * (int)sizeof(RED) : 0);

    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    unsigned char *sData = smem;
    ACC *sW = reinterpret_cast<ACC *>(smem + SM.off_w);
    RED *red = reinterpret_cast<RED *>(smem + SM.off_red);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + SM.off_bar);
    uint64_t *empty = full + STAGES;
    volatile int *tile_q = reinterpret_cast<volatile int *>(empty + STAGES);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t row_bytes = p.HW * (int64_t)sizeof(T);
    const int n_tiles = (int)((row_bytes + SEG - 1) / SEG);
    // the window is at most two runs of consecutive slots of the frame store (a ring wraps once)
    const int run0 = min(p.n, p.cap - p.slot0), run1 = p.n - run0;

    if (threadIdx.x == 0) {
        for (int i = 0; i < STAGES; ++i) {
            mbar_init(&full[i], 2);          // the producer's expect_tx arrival + its "weights written" arrival
            mbar_init(&empty[i], NW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == 0) {
        // ===== producer: TMA boxes + weight rows, tile scheduler =====
        const ACC *wtab = static_cast<const ACC *>(p.wtab);
        int stage = 0, it = 0;
        uint32_t phase = 0;
        for (;; ++it) {
            int tile = 0;
            if (lane == 0) {
                tile = (int)atomicAdd(tile_counter, 1u);
                if (tile >= n_tiles) tile = -1;
                tile_q[it & (TQ - 1)] = tile;            // published by the arrivals on full[stage] below
            }
            tile = __shfl_sync(0xffffffffu, tile, 0);
            if (tile < 0) {
                if (lane == 0) {
                    mbar_wait(&empty[stage], phase ^ 1);
                    mbar_arrive(&full[stage]);
                    mbar_arrive(&full[stage]);
                }
                break;
            }
            int fi = 0;                                    // frame index inside the window of the chunk's first frame
            for (int run = 0; run < 2; ++run) {
                const int rn = run ? run1 : run0, rslot = run ? 0 : p.slot0;
                for (int c0 = 0; c0 < rn; c0 += KC) {
                    const int nf = min(KC, rn - c0);
                    mbar_wait(&empty[stage], phase ^ 1);
                    if (lane == 0) {
                        mbar_expect_tx(&full[stage], (uint32_t)SM.data_stage);
                        // rows beyond the store are zero filled, rows beyond the run are never used
                        tma_load_2d(sData + (size_t)stage * SM.data_stage, &tmap, &full[stage], tile * (SEG / 8), rslot + c0,
                                    0x12F0000000000000ull /* evict first: every sample is read once */);
                    }
                    ACC *wdst = sW + (size_t)stage * KC * ROWS;
                    for (int i = lane; i < nf * ROWS; i += 32) {
                        int e = p.w0 + fi + i / ROWS;
                        if (e >= p.cap_w) e -= p.cap_w;
                        wdst[i] = __ldg(wtab + (int64_t)e * ROWS + (i % ROWS));
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&full[stage]);
                    fi += nf;
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
            }
        }
        return;
    }

    // ===== consumers =====
    const int cw = warp - 1, cg = cw % CG, ts = cw / CG;
    const int col = (cg * 32 + lane) * VB;                 // byte offset of this thread's pixels inside the segment
    const int tcol = cg * 32 + lane;                       // thread column inside the tile
    int stage = 0;
    uint32_t phase = 0;
    for (int it = 0;; ++it) {
        mbar_wait(&full[stage], phase);
        const int tile = tile_q[it & (TQ - 1)];
        if (tile < 0) break;
        const int64_t pix0 = ((int64_t)tile * SEG + col) / (int64_t)sizeof(T);
        const bool active = pix0 < p.HW;

        ACC acc[ROWS][V];
#pragma unroll
        for (int r = 0; r < ROWS; ++r)
#pragma unroll
            for (int v = 0; v < V; ++v) acc[r][v] = 0;
        float pedm[V];
#pragma unroll
        for (int v = 0; v < V; ++v) pedm[v] = 8388608.0f;

        bool first = true;
        for (int run = 0; run < 2; ++run) {
            const int rn = run ? run1 : run0;
            for (int c0 = 0; c0 < rn; c0 += KC) {
                const int nf = min(KC, rn - c0);
                if (!first) mbar_wait(&full[stage], phase);
                const unsigned char *d = sData + (size_t)stage * SM.data_stage + col;
                const ACC *wrow = sW + (size_t)stage * KC * ROWS;
                if (first) {
                    first = false;
                    if constexpr (!IS_INT) {
                        // pedestal = the pixel's first sample in the window (exact integer), DESIGN.md "Precision"
                        uint32_t w0[PX::NW];
                        PX::load_shared(d, w0);
#pragma unroll
                        for (int v = 0; v < V; ++v) pedm[v] = PX::getf_biased(w0, v);
                    }
                }
                int f = ts;
                if (nf == KC) {
                    // full stage: four frames per step (KC / TS is a multiple of 4)
                    for (; f < KC; f += 4 * TS) {
                        uint32_t w[4][PX::NW];
                        ACC wt[4][ROWS];
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            PX::load_shared(d + (size_t)(f + u * TS) * SEG, w[u]);
                            load_weights_shared<ACC, ROWS>(wrow + (f + u * TS) * ROWS, wt[u]);
                        }
#pragma unroll
                        for (int u = 0; u < 4; ++u) accumulate<T, ACC, ROWS, V>(w[u], wt[u], pedm, acc);
                    }
                } else {
                    for (; f < nf; f += TS) {
                        uint32_t w[PX::NW];
                        ACC wt[ROWS];
                        PX::load_shared(d + (size_t)f * SEG, w);
                        load_weights_shared<ACC, ROWS>(wrow + f * ROWS, wt);
                        accumulate<T, ACC, ROWS, V>(w, wt, pedm, acc);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[stage]);
                if (++stage == STAGES) { stage = 0; phase ^= 1; }
            }
        }

        // ---- combine the TS time slices (fp64 / int32), then A4 ----
        if (TS > 1) {
            for (int yy = 0; yy < TS; ++yy) {
                if (ts == yy) {
#pragma unroll
                    for (int r = 0; r < ROWS; ++r)
#pragma unroll
                        for (int v = 0; v < V; ++v) {
                            RED *cell = &red[(r * V + v) * (CG * 32) + tcol];
                            if (yy == 0) *cell = (RED)acc[r][v];
                            else *cell += (RED)acc[r][v];
                        }
                }
                named_barrier(1, NW * 32);
            }
        }
        if (active) {
            for (int v = ts; v < V; v += TS) {
                const int64_t pixel = pix0 + v;
                double val[ROWS];
                RED a[ROWS];
                if (TS > 1) {
#pragma unroll
                    for (int r = 0; r < ROWS; ++r) a[r] = red[(r * V + v) * (CG * 32) + tcol];
                } else {
#pragma unroll
                    for (int r = 0; r < ROWS; ++r) {
                        // v is a runtime index: select without forcing acc[][] into local memory
                        RED t = 0;
#pragma unroll
                        for (int vv = 0; vv < V; ++vv) t = (vv == v) ? (RED)acc[r][vv] : t;
                        a[r] = t;
                    }
                }
                if constexpr (IS_INT) {
#pragma unroll
                    for (int r = 0; r < ROWS; ++r) {
                        val[r] = (double)a[r];
                        if (p.acc_out) static_cast<int *>(p.acc_out)[(int64_t)r * p.HW + pixel] = a[r];
                    }
                } else {
                    float pm = 0.f;
#pragma unroll
                    for (int vv = 0; vv < V; ++vv) pm = (vv == v) ? pedm[vv] : pm;
                    const double ped = (double)(pm - 8388608.0f);
#pragma unroll
                    for (int r = 0; r < ROWS; ++r) {
                        if (p.acc_out) static_cast<double *>(p.acc_out)[(int64_t)r * p.HW + pixel] = a[r];
                        const double wsum = p.cum[(int64_t)p.cum_hi * ROWS + r] - p.cum[(int64_t)p.cum_lo * ROWS + r];
                        val[r] = a[r] + ped * wsum;     // sum x w = sum (x - ped) w + ped * sum w
                    }
                    if (p.ped_out) p.ped_out[pixel] = (float)ped;
                }
                finalise_pixel<ROWS>(p.fin, val, pixel, p.HW);
            }
        }
        if (TS > 1) named_barrier(1, NW * 32);              // red is free for the next tile
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int red_bytes_for(int seg, int vb, int rows, int v, bool is_int)
{
    const int cg = seg / (32 * vb), ts = NW / cg;
    return ts > 1 ? rows * v * cg * 32 * (is_int ? 4 : 8) : 0;
}

template <typename T, typename ACC, int ROWS>
cudaError_t launch_stream_t(const void *tmap, const DemodParams &p, const StreamShape &sh, unsigned int *counter, int n_sms, cudaStream_t st)
{
    constexpr int V = pick_v(sizeof(T), ROWS);
    constexpr bool IS_INT = std::is_same<ACC, int>::value;
    const StreamSmem SM(sh.seg, sh.kc, sh.stages, ROWS, red_bytes_for(sh.seg, V * (int)sizeof(T), ROWS, V, IS_INT));
    auto kern = k_demod_stream<T, ACC, ROWS, V>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SM.total + 128);
    if (e != cudaSuccess) return e;
    const int64_t row_bytes = p.HW * (int64_t)sizeof(T);
    const int n_tiles = (int)((row_bytes + sh.seg - 1) / sh.seg);
    e = cudaMemsetAsync(counter, 0, sizeof(unsigned int), st);
    if (e != cudaSuccess) return e;
    kern<<<n_tiles < n_sms ? n_tiles : n_sms, 32 * (NW + 1), SM.total + 128, st>>>(*reinterpret_cast<const CUtensorMap *>(tmap), p, sh, counter);
    return cudaGetLastError();
}

template <typename T, typename ACC>
cudaError_t launch_stream_r(int rows, const void *tmap, const DemodParams &p, const StreamShape &sh, unsigned int *counter, int n_sms, cudaStream_t st)
{
    switch (rows) {
    case 2: return launch_stream_t<T, ACC, 2>(tmap, p, sh, counter, n_sms, st);
    case 4: return launch_stream_t<T, ACC, 4>(tmap, p, sh, counter, n_sms, st);
    case 8: return launch_stream_t<T, ACC, 8>(tmap, p, sh, counter, n_sms, st);
    case 16: return launch_stream_t<T, ACC, 16>(tmap, p, sh, counter, n_sms, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace

// Tile shape for this (dtype, rows, frame size), or seg = 0 when the streaming kernel does not apply (row pitch or
// base not 16-byte aligned, or a frame too small to give every SM a tile: k_demod_whole handles those).
StreamShape qld_stream_shape(int dtype, int is_int, int rows, int64_t HW, const void *frames, int n_sms)
{
    StreamShape sh = {0, 0, 0};
    const int bytes = dtype == QLD_U8 ? 1 : 2;
    const int v = pick_v(bytes, rows), vb = v * bytes;
    const int64_t row_bytes = HW * bytes;
    if (row_bytes % 16 != 0 || (reinterpret_cast<uintptr_t>(frames) & 15) != 0) return sh;
    int seg = 2048;                                        // TMA box: at most 256 8-byte elements per row
    if (seg > NW * 32 * vb) seg = NW * 32 * vb;
    while (seg > 32 * vb && (row_bytes + seg - 1) / seg < 4 * (int64_t)n_sms) seg /= 2;
    int kc = 16, stages = 0;
    bool forced = false;
    if (const char *e = getenv("QLD_STREAM_TILE")) {      // tuning / test override: "SEG,KC" (also lifts the size threshold)
        int s2 = 0, k2 = 0;
        if (sscanf(e, "%d,%d", &s2, &k2) == 2 && s2 >= 32 * vb && s2 <= NW * 32 * vb && s2 <= 2048 && (s2 & (s2 - 1)) == 0 && k2 >= 4 && k2 <= 256) { seg = s2; kc = k2; forced = true; }
    }
    if (!forced && (row_bytes + seg - 1) / seg < n_sms) return sh;
    const int ts = NW / (seg / (32 * vb));
    if (kc < 4 * ts) kc = 4 * ts;                          // every slice gets a multiple of four frames per stage
    kc = (kc + 4 * ts - 1) / (4 * ts) * (4 * ts);
    const int red = red_bytes_for(seg, vb, rows, v, is_int != 0);
    stages = (int)((200 * 1024 - red) / (seg * kc + kc * rows * 4));
    if (stages > 12) stages = 12;
    if (stages < 2) return StreamShape{0, 0, 0};
    sh.seg = seg; sh.kc = kc; sh.stages = stages;
    return sh;
}

// 2-D tensor map over the frame store viewed as [cap frames][row_bytes / 8] 8-byte elements, box {seg / 8, kc}.
cudaError_t qld_stream_encode_tmap(void *tmap_out, const void *frames, int64_t row_bytes, int cap, const StreamShape &sh)
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *sym = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres);
        if (e != cudaSuccess) return e;
        if (!sym || qres != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
        fn = reinterpret_cast<EncodeTiledFn>(sym);
    }
    const cuuint64_t dims[2] = {(cuuint64_t)(row_bytes / 8), (cuuint64_t)cap};
    const cuuint64_t strides[1] = {(cuuint64_t)row_bytes};
    const cuuint32_t box[2] = {(cuuint32_t)(sh.seg / 8), (cuuint32_t)sh.kc};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(reinterpret_cast<CUtensorMap *>(tmap_out), CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void *>(frames), dims, strides, box,
                    estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

cudaError_t qld_launch_demod_stream(int dtype, int is_int, int rows, const void *tmap, const DemodParams &p, const StreamShape &sh,
                                    unsigned int *counter, int n_sms, cudaStream_t st)
{
    if (dtype == QLD_U8)
        return is_int ? launch_stream_r<uint8_t, int>(rows, tmap, p, sh, counter, n_sms, st) : launch_stream_r<uint8_t, float>(rows, tmap, p, sh, counter, n_sms, st);
    return is_int ? launch_stream_r<uint16_t, int>(rows, tmap, p, sh, counter, n_sms, st) : launch_stream_r<uint16_t, float>(rows, tmap, p, sh, counter, n_sms, st);
}

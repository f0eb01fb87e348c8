// Sliding-window update ("sliding sequence") for frames large enough to give every
// SM a tile: the hop's new frames (and, without per-batch partial sums, the expired ones with weight -w) are added to the
// sums the previous window left in HBM, and A4 runs on the updated sums.
//
// A hop is short (32 frames on BASELINE.json configs[3]), so per pixel the launch moves as many bytes of STATE -- stored
// sums, the expired batch's partial sums, the map -- as of frames, and in round 1 the threads that fetched that state with
// ordinary loads sat on the DRAM latency once per tile (0.52 of the HBM roof).  Here no thread ever waits on global memory:
//
//   warp 0      producer   TMA boxes {SEG bytes} x {KC frames} of the run list into a ring of stages (as k_demod_stream),
//                          and, per tile, 1-D bulk copies of the tile's state rows into one of NSB state buffers,
//                          one to two tiles ahead;
//   warps 1..8  consumers  thread = 4 adjacent pixels, ALL frames of the launch (no time slices, nothing to combine):
//                          LDS -> byte-permute -> integer add / FFMA2; then the update and A4 out of the state buffer, the
//                          results written back INTO the state buffer;
//   warp 9      store      bulk copies shared -> global of the updated rows and the map rows, then hands the buffer back.
//
// Arithmetic is that of k_demod_stream / k_demod_slide: int32 bins exact; fp32 partial sums of pedestal-subtracted samples
// added into fp64 stored sums.
#include <string.h>

#include "qld_device.cuh"
#include "qld_ptx.cuh"
#include "qld_slide.h"

using namespace qld_dev;
using namespace qld_ptx;

namespace {

constexpr int SL_NW = 8;                  // consumer warps
constexpr int SL_V = 4;                   // pixels per consumer thread
constexpr int SL_TP = SL_NW * 32 * SL_V;  // pixels per tile (1024)
constexpr int SL_TQ = 16;                 // tile-id queue entries (the producer runs at most `stages` <= 12 chunks ahead)
constexpr int SL_MAX_SB = 4;
constexpr int SL_THREADS = 32 * (SL_NW + 2);

// bulk copy shared -> global, tracked by the issuing thread's bulk async-group
__device__ __forceinline__ void bulk_store(void *dst_global, const void *src_shared, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_global), "r"(smem_u32(src_shared)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// integer dot products of packed samples with packed signed 8-bit weights (exact, s32 accumulate):
//   dp2a: two unsigned 16-bit samples (the same pixel in two consecutive frames) x weight bytes 0, 1
//   dp4a: four unsigned 8-bit samples (four consecutive frames) x weight bytes 0..3
__device__ __forceinline__ int dp2a_u16_s8(uint32_t a, int b, int c)
{
    int d;
    asm("dp2a.lo.u32.s32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
__device__ __forceinline__ int dp4a_u8_s8(uint32_t a, int b, int c)
{
    int d;
    asm("dp4a.u32.s32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

// shared-memory carve-up.  A state buffer holds, for the TP pixels of a tile, rows of TP cells:
//   acc[ROWS] (RED), part[ROWS] (RED, block-partial mode), ped (float, fp32 mode), maps[n_map_rows] (float)
struct SlideSmem {
    int data_stage, w_stage, state_bytes, off_acc, off_part, off_ped, off_map, off_w, off_state, off_bar, total;
    __host__ __device__ SlideSmem(int seg, int kc, int stages, int nsb, int rows, int red_size, bool part, bool has_ped, int n_map_rows)
    {
        data_stage = seg * kc;
        w_stage = kc * 4 * 4;             // fp32: [KC][ROWS] floats; integer bins: [KC / G][4] words of G packed signed bytes
        off_acc = 0;
        off_part = off_acc + rows * SL_TP * red_size;
        off_ped = off_part + (part ? rows * SL_TP * red_size : 0);
        off_map = off_ped + (has_ped ? SL_TP * 4 : 0);
        state_bytes = off_map + n_map_rows * SL_TP * 4;
        off_w = stages * data_stage;
        off_state = (off_w + stages * w_stage + 127) & ~127;
        off_bar = off_state + nsb * state_bytes;
        total = off_bar + (2 * stages + 3 * SL_MAX_SB) * 8 + SL_TQ * 4 + SL_MAX_SB * 4 + 16;
    }
};


template <typename T, typename ACC, int ROWS, bool PART>
__global__ void __launch_bounds__(SL_THREADS, 1)
k_slide_bulk(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ DemodParams p, const SlideShape sh, const int n_map_rows,
             unsigned int *tile_counter, unsigned int *counter_next)
{
    using PX = Pix<T, SL_V>;
    // ACC = float: fp32 partial sums of pedestal-subtracted samples, fp64 stored sums;  ACC = int: integer phase bins (exact);
    // ACC = long long: Q1.30 fixed-point references, exact int64 sums (drift-free sliding at any nu)
    constexpr bool IS_INT = std::is_same<ACC, int>::value;
    constexpr bool IS_FIX = std::is_same<ACC, long long>::value;
    constexpr bool IS_F32 = std::is_same<ACC, float>::value;
    using WT = typename std::conditional<IS_F32, float, int>::type;                        // weight table entries
    using RED = typename std::conditional<IS_F32, double, ACC>::type;                      // stored sums
    constexpr int V = SL_V, TP = SL_TP;
    constexpr int VB = V * (int)sizeof(T);

    const int SEG = sh.seg, KC = sh.kc, STAGES = sh.stages, NSB = sh.nsb;
    const SlideSmem SM(SEG, KC, STAGES, NSB, ROWS, (int)sizeof(RED), PART, IS_F32, n_map_rows);

    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    unsigned char *sData = smem;
    unsigned char *sState = smem + SM.off_state;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + SM.off_bar);
    uint64_t *empty = full + STAGES;
    uint64_t *state_full = empty + STAGES;                 // [NSB] producer's bulk copies have landed
    uint64_t *out_full = state_full + SL_MAX_SB;           // [NSB] consumers have written the updated rows
    uint64_t *state_empty = out_full + SL_MAX_SB;          // [NSB] the store warp's copies have read the buffer
    volatile int *tile_q = reinterpret_cast<volatile int *>(state_empty + SL_MAX_SB);
    volatile int *out_tile = tile_q + SL_TQ;               // [NSB] tile whose results sit in the buffer

    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
    const int64_t row_bytes = p.HW * (int64_t)sizeof(T);
    const int n_tiles = (int)((p.HW + TP - 1) / TP);
    int n_chunks = 0;                                      // pipeline stages per tile
    for (int run = 0; run < p.n_runs; ++run) n_chunks += (p.run[run].n + KC - 1) / KC;

    if (threadIdx.x == 0) {
        if (blockIdx.x == 0) {
            *counter_next = 0;                    // the next launch's tile counter (three rotate: no memset between launches)
            __threadfence();
        }
    }
    if (warp == 0) {
        // barrier initialisation spread over the lanes of warp 0 (a serial loop in one thread cost 0.5 us of every launch)
        const int n_bar = 2 * STAGES + 3 * SL_MAX_SB;
        for (int i = lane; i < n_bar; i += 32) {
            uint32_t count;
            if (i < STAGES) count = 2;                                   // full: the producer's expect_tx arrival + its "weights written" arrival
            else if (i < 2 * STAGES) count = SL_NW;                      // empty
            else {
                const int j = (i - 2 * STAGES) / SL_MAX_SB;              // state_full, out_full, state_empty
                count = j == 1 ? SL_NW * 32 : 1;
            }
            mbar_init(&full[i], count);                                  // the barriers are contiguous: full, empty, state_full, out_full, state_empty
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    (void)row_bytes;
    // Programmatic dependent launch: the next launch of the stream may start on SMs as they free up -- its CTAs initialise their
    // barriers and put the frames of their first tile in flight while this launch drains -- but it touches the sums this launch
    // updates only after griddepcontrol.wait (producer, below), i.e. after this grid has completed and its writes are visible.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    RED *accg = static_cast<RED *>(p.acc_out);
    RED *partg = static_cast<RED *>(p.part);

    if (warp == 0) {
        // ===== producer: tile scheduler, state rows (bulk copies), frame boxes (TMA) + weight rows =====
        const WT *wtab = static_cast<const WT *>(p.wtab);
        int stage = 0;
        uint32_t phase = 0;
        int next = (int)blockIdx.x;
        for (int it = 0;; ++it) {
            int tile = 0;
            if (lane == 0) {
                tile = next < n_tiles ? next : -1;
                if (tile >= 0) next = (int)gridDim.x + (int)atomicAdd(tile_counter, 1u);
                tile_q[it & (SL_TQ - 1)] = tile;             // published by the arrivals on full[stage] below
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
            // the tile's state: previous sums, the expired batch's partial sums, the pedestal
            const int sb = it % NSB;
            const int64_t pix0 = (int64_t)tile * TP;
            const int npx = (int)min((int64_t)TP, p.HW - pix0);
            // The first tile's frames do not depend on the launch before this one, its state does: when all of the tile's stages
            // fit the (still empty) ring, the frames go in flight first and the dependency wait + state copies follow, so that
            // the ramp-up of this launch overlaps the tail of the previous one (programmatic dependent launch).
            const bool late_state = it == 0 && n_chunks <= STAGES;
            auto issue_state = [&]() {
            if (lane == 0) {
                if (it == 0) asm volatile("griddepcontrol.wait;" ::: "memory");   // the previous launch's sums are final from here on
                mbar_wait(&state_empty[sb], (uint32_t)((it / NSB) & 1) ^ 1u);
                unsigned char *st = sState + (size_t)sb * SM.state_bytes;
                const uint32_t rb = (uint32_t)(npx * (int)sizeof(RED));
                uint32_t bytes = (uint32_t)ROWS * rb * (PART ? 2u : 1u) + (IS_F32 ? (uint32_t)(npx * 4) : 0u);
                mbar_expect_tx(&state_full[sb], bytes);
#pragma unroll
                for (int r = 0; r < ROWS; ++r) {
                    bulk_load(st + SM.off_acc + (size_t)r * TP * sizeof(RED), accg + (int64_t)r * p.HW + pix0, rb, &state_full[sb]);
                    if (PART) bulk_load(st + SM.off_part + (size_t)r * TP * sizeof(RED), partg + (int64_t)r * p.HW + pix0, rb, &state_full[sb]);
                }
                if (IS_F32) bulk_load(st + SM.off_ped, p.ped_in + pix0, (uint32_t)(npx * 4), &state_full[sb]);
            }
            };
            if (!late_state) issue_state();
            for (int run = 0; run < p.n_runs; ++run) {
                const int rn = p.run[run].n, rslot = p.run[run].slot0, rw0 = p.run[run].w0;
                const WT sgn = (WT)p.run[run].sign;
                for (int c0 = 0; c0 < rn; c0 += KC) {
                    const int nf = min(KC, rn - c0);
                    mbar_wait(&empty[stage], phase ^ 1);
                    if (lane == 0) {
                        mbar_expect_tx(&full[stage], (uint32_t)SM.data_stage);
                        // rows beyond the store are zero filled, rows beyond the run are never used
                        tma_load_2d(sData + (size_t)stage * SM.data_stage, &tmap, &full[stage], tile * (SEG / 8), rslot + c0,
                                    0x12F0000000000000ull /* evict first: every sample is read once */);
                    }
                    if constexpr (IS_INT) {
                        // word (q, r) = the weights of row r for the G frames q*G .. q*G+G-1 of the stage as signed bytes
                        // (zero beyond the run and for padding rows: integer 0 * anything = 0)
                        constexpr int G = 4 / (int)sizeof(T);
                        int *wdst = reinterpret_cast<int *>(smem + SM.off_w + (size_t)stage * SM.w_stage);
                        for (int i = lane; i < (KC / G) * 4; i += 32) {
                            const int q = i >> 2, r = i & 3;
                            uint32_t word = 0;
                            if (r < ROWS) {
#pragma unroll
                                for (int b = 0; b < G; ++b) {
                                    const int fr = q * G + b;
                                    if (fr < nf) {
                                        int e = rw0 + c0 + fr;
                                        if (e >= p.cap_w) e -= p.cap_w;
                                        word |= (uint32_t)((sgn * __ldg(wtab + (int64_t)e * ROWS + r)) & 0xff) << (8 * b);
                                    }
                                }
                            }
                            wdst[i] = (int)word;
                        }
                    } else {
                        WT *wdst = reinterpret_cast<WT *>(smem + SM.off_w + (size_t)stage * SM.w_stage);
                        for (int i = lane; i < nf * ROWS; i += 32) {
                            int e = rw0 + c0 + i / ROWS;
                            if (e >= p.cap_w) e -= p.cap_w;
                            wdst[i] = sgn * __ldg(wtab + (int64_t)e * ROWS + (i % ROWS));
                        }
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&full[stage]);
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
            }
            if (late_state) issue_state();
        }
        return;
    }

    // row index of map `which` (0 = I, 1 = Q, 2 = amplitude, 3 = phase) of reference k inside the state buffer, -1: not requested
    float *const map_ptr[4] = {p.fin.I, p.fin.Q, p.fin.amp, p.fin.phase};
    int map_slot[4], n_which = 0;
#pragma unroll
    for (int w = 0; w < 4; ++w) map_slot[w] = map_ptr[w] ? n_which++ : -1;

    if (warp == SL_NW + 1) {
        // ===== store warp: updated rows and maps, shared -> global, then the buffer goes back to the producer =====
        for (int it = 0;; ++it) {
            const int sb = it % NSB;
            mbar_wait(&out_full[sb], (uint32_t)((it / NSB) & 1));
            const int tile = out_tile[sb];
            if (tile < 0) break;
            if (lane == 0) {
                unsigned char *st = sState + (size_t)sb * SM.state_bytes;
                const int64_t pix0 = (int64_t)tile * TP;
                const int npx = (int)min((int64_t)TP, p.HW - pix0);
                const uint32_t rb = (uint32_t)(npx * (int)sizeof(RED));
#pragma unroll
                for (int r = 0; r < ROWS; ++r) {
                    bulk_store(accg + (int64_t)r * p.HW + pix0, st + SM.off_acc + (size_t)r * TP * sizeof(RED), rb);
                    if (PART) bulk_store(partg + (int64_t)r * p.HW + pix0, st + SM.off_part + (size_t)r * TP * sizeof(RED), rb);
                }
                for (int k = 0; k < p.fin.K; ++k)
#pragma unroll
                    for (int w = 0; w < 4; ++w)
                        if (map_slot[w] >= 0)
                            bulk_store(map_ptr[w] + (int64_t)k * p.HW + pix0, st + SM.off_map + (size_t)(k * n_which + map_slot[w]) * TP * 4, (uint32_t)(npx * 4));
                bulk_commit();
                bulk_wait_read0();                         // the copies have read the buffer (their global writes may still be in flight)
                mbar_arrive(&state_empty[sb]);
            }
            __syncwarp();
        }
        if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
        return;
    }

    // ===== consumers =====
    const int ct = (int)threadIdx.x - 32;                  // consumer thread: pixels 4*ct .. 4*ct+3 of the tile
    const uint32_t bsw = p.big_endian ? 0x11u : 0u;
    // dp2a operands: (pixel v of frame f, of frame f+1) as two 16-bit halves; QLD_U16_BE swaps the bytes of each half
    const uint32_t sel_lo = p.big_endian ? 0x4501u : 0x5410u, sel_hi = p.big_endian ? 0x6723u : 0x7632u;
    double wsum[ROWS];
#pragma unroll
    for (int r = 0; r < ROWS; ++r) wsum[r] = 0.0;
    if constexpr (IS_F32) {
#pragma unroll
        for (int r = 0; r < ROWS; ++r) wsum[r] = p.cum[(int64_t)p.cum_hi * ROWS + r] - p.cum[(int64_t)p.cum_lo * ROWS + r];
    }
    const FinParams &f = p.fin;
    int stage = 0;
    uint32_t phase = 0;
    for (int it = 0;; ++it) {
        mbar_wait(&full[stage], phase);
        const int tile = tile_q[it & (SL_TQ - 1)];
        const int sb = it % NSB;
        const uint32_t spar = (uint32_t)((it / NSB) & 1);
        if (tile < 0) {
            // end of work: tell the store warp, once it is done with this buffer's previous tile
            mbar_wait(&state_empty[sb], spar ^ 1u);
            if (ct == 0) out_tile[sb] = -1;
            mbar_arrive(&out_full[sb]);
            break;
        }
        unsigned char *st = sState + (size_t)sb * SM.state_bytes;

        ACC acc[ROWS][V];
#pragma unroll
        for (int r = 0; r < ROWS; ++r)
#pragma unroll
            for (int v = 0; v < V; ++v) acc[r][v] = 0;
        float pedm[V], pedf[V];
#pragma unroll
        for (int v = 0; v < V; ++v) { pedm[v] = 8388608.0f; pedf[v] = 0.0f; }
        if constexpr (IS_F32) {
            // the pedestal the stored sums were seeded with (exact integer) is needed before the first frame
            mbar_wait(&state_full[sb], spar);
            const float4 pd = *reinterpret_cast<const float4 *>(st + SM.off_ped + (size_t)ct * 16);
            pedf[0] = pd.x; pedf[1] = pd.y; pedf[2] = pd.z; pedf[3] = pd.w;
#pragma unroll
            for (int v = 0; v < V; ++v) pedm[v] = 8388608.0f + pedf[v];
        }

        // ---- frame loop: every consumer thread takes every frame of the launch for its 4 pixels ----
        bool first = true;
        for (int run = 0; run < p.n_runs; ++run) {
            const int rn = p.run[run].n;
            for (int c0 = 0; c0 < rn; c0 += KC) {
                const int nf = min(KC, rn - c0);
                if (!first) mbar_wait(&full[stage], phase);
                first = false;
                const unsigned char *d = sData + (size_t)stage * SM.data_stage + (size_t)ct * VB;
                if constexpr (IS_INT) {
                    // G consecutive frames of a pixel packed into one register (byte permutes), one dot-product instruction
                    // per pixel, row and frame group
                    constexpr int G = 4 / (int)sizeof(T);
                    const int4 *wq = reinterpret_cast<const int4 *>(smem + SM.off_w + (size_t)stage * SM.w_stage);
                    const int ng = (nf + G - 1) / G;
#pragma unroll 2
                    for (int q = 0; q < ng; ++q) {
                        const int4 wt4 = wq[q];
                        const int wt[4] = {wt4.x, wt4.y, wt4.z, wt4.w};
                        uint32_t px[V];
                        if constexpr (sizeof(T) == 2) {
                            const uint2 f0 = *reinterpret_cast<const uint2 *>(d + (size_t)(2 * q) * SEG);
                            const uint2 f1 = *reinterpret_cast<const uint2 *>(d + (size_t)(2 * q + 1) * SEG);
                            px[0] = __byte_perm(f0.x, f1.x, sel_lo);
                            px[1] = __byte_perm(f0.x, f1.x, sel_hi);
                            px[2] = __byte_perm(f0.y, f1.y, sel_lo);
                            px[3] = __byte_perm(f0.y, f1.y, sel_hi);
#pragma unroll
                            for (int r = 0; r < ROWS; ++r)
#pragma unroll
                                for (int v = 0; v < V; ++v) acc[r][v] = dp2a_u16_s8(px[v], wt[r], acc[r][v]);
                        } else {
                            uint32_t fw[4];
#pragma unroll
                            for (int b = 0; b < 4; ++b) fw[b] = *reinterpret_cast<const uint32_t *>(d + (size_t)(4 * q + b) * SEG);
                            // 4 x 4 byte transpose: px[v] = bytes v of the four frames
                            const uint32_t t0 = __byte_perm(fw[0], fw[1], 0x5140), t1 = __byte_perm(fw[0], fw[1], 0x7362);
                            const uint32_t t2 = __byte_perm(fw[2], fw[3], 0x5140), t3 = __byte_perm(fw[2], fw[3], 0x7362);
                            px[0] = __byte_perm(t0, t2, 0x5410);
                            px[1] = __byte_perm(t0, t2, 0x7632);
                            px[2] = __byte_perm(t1, t3, 0x5410);
                            px[3] = __byte_perm(t1, t3, 0x7632);
#pragma unroll
                            for (int r = 0; r < ROWS; ++r)
#pragma unroll
                                for (int v = 0; v < V; ++v) acc[r][v] = dp4a_u8_s8(px[v], wt[r], acc[r][v]);
                        }
                    }
                } else if constexpr (IS_FIX) {
                    // exact: unsigned sample times Q1.30 reference, 64-bit multiply-add
                    const int *wrow = reinterpret_cast<const int *>(smem + SM.off_w + (size_t)stage * SM.w_stage);
#pragma unroll 4
                    for (int fr = 0; fr < nf; ++fr) {
                        uint32_t w[PX::NW];
                        int wt[ROWS];
                        PX::load_shared(d + (size_t)fr * SEG, w);
                        load_weights_shared<int, ROWS>(wrow + fr * ROWS, wt);
#pragma unroll
                        for (int v = 0; v < V; ++v) {
                            const long long x = (long long)PX::geti(w, v, bsw);
#pragma unroll
                            for (int r = 0; r < ROWS; ++r) acc[r][v] += x * (long long)wt[r];
                        }
                    }
                } else {
                    const ACC *wrow = reinterpret_cast<const ACC *>(smem + SM.off_w + (size_t)stage * SM.w_stage);
                    int fr = 0;
                    for (; fr + 4 <= nf; fr += 4) {
                        uint32_t w[4][PX::NW];
                        ACC wt[4][ROWS];
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            PX::load_shared(d + (size_t)(fr + u) * SEG, w[u]);
                            load_weights_shared<ACC, ROWS>(wrow + (fr + u) * ROWS, wt[u]);
                        }
#pragma unroll
                        for (int u = 0; u < 4; ++u) accumulate<T, ACC, ROWS, V>(w[u], wt[u], pedm, acc, bsw);
                    }
                    for (; fr < nf; ++fr) {
                        uint32_t w[PX::NW];
                        ACC wt[ROWS];
                        PX::load_shared(d + (size_t)fr * SEG, w);
                        load_weights_shared<ACC, ROWS>(wrow + fr * ROWS, wt);
                        accumulate<T, ACC, ROWS, V>(w, wt, pedm, acc, bsw);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[stage]);
                if (++stage == STAGES) { stage = 0; phase ^= 1; }
            }
        }

        // ---- update the stored sums (A5) in place in the state buffer, then A4 ----
        if constexpr (!IS_F32) mbar_wait(&state_full[sb], spar);
        RED a[ROWS][V];
#pragma unroll
        for (int r = 0; r < ROWS; ++r) {
            RED *arow = reinterpret_cast<RED *>(st + SM.off_acc) + (size_t)r * TP + (size_t)ct * V;
            RED old[V];
            load_vec<RED, V>(arow, old);
            RED mine[V];
#pragma unroll
            for (int v = 0; v < V; ++v) mine[v] = (RED)acc[r][v];
            if constexpr (PART) {
                // 8(f3): this launch's sums replace the expired batch's partial sums
                RED *prow = reinterpret_cast<RED *>(st + SM.off_part) + (size_t)r * TP + (size_t)ct * V;
                RED exp[V];
                load_vec<RED, V>(prow, exp);
                store_vec<RED, V>(prow, mine);
#pragma unroll
                for (int v = 0; v < V; ++v) a[r][v] = old[v] - exp[v] + mine[v];
            } else {
#pragma unroll
                for (int v = 0; v < V; ++v) a[r][v] = old[v] + mine[v];
            }
            store_vec<RED, V>(arow, a[r]);
        }
        for (int k = 0; k < f.K; ++k) {
            float o[4][V];
#pragma unroll
            for (int v = 0; v < V; ++v) {
                double S = 0.0, C = 0.0;
                if constexpr (IS_INT) {
                    const int off = f.row_off[k], end = off + f.n_rows[k];
#pragma unroll
                    for (int r = 0; r < ROWS; ++r)
                        if (r >= off && r < end) {
                            S = fma((double)a[r][v], f.sw[r], S);
                            C = fma((double)a[r][v], f.cw[r], C);
                        }
                } else if constexpr (IS_FIX) {
#pragma unroll
                    for (int r = 0; r + 1 < ROWS; r += 2)
                        if (r == 2 * k) {
                            S = (double)a[r][v] * 9.31322574615478515625e-10;         // 2^-30
                            C = (double)a[r + 1][v] * 9.31322574615478515625e-10;
                        }
                } else {
#pragma unroll
                    for (int r = 0; r + 1 < ROWS; r += 2)
                        if (r == 2 * k) {
                            S = (double)a[r][v] + (double)pedf[v] * wsum[r];          // sum x w = sum (x - ped) w + ped * sum w
                            C = (double)a[r + 1][v] + (double)pedf[v] * wsum[r + 1];
                        }
                }
                rotate_iq(f.rot, k, S, C);
                S *= f.scale;
                C *= f.scale;
                o[0][v] = (float)S;
                o[1][v] = (float)C;
                o[2][v] = map_slot[2] >= 0 ? (float)sqrt(S * S + C * C) : 0.0f;
                o[3][v] = (map_slot[3] >= 0 && !(S == 0.0 && C == 0.0)) ? (float)atan2(C, S) : 0.0f;
            }
#pragma unroll
            for (int w = 0; w < 4; ++w)
                if (map_slot[w] >= 0)
                    store_vec<float, V>(reinterpret_cast<float *>(st + SM.off_map) + (size_t)(k * n_which + map_slot[w]) * TP + (size_t)ct * V, o[w]);
        }
        fence_async_smem();                                // generic-proxy writes before the store warp's bulk copies read them
        if (ct == 0) out_tile[sb] = tile;
        mbar_arrive(&out_full[sb]);
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

template <typename T, typename ACC, int ROWS, bool PART>
cudaError_t launch_slide_n(const void *tmap, const DemodParams &p, const SlideShape &sh, int n_map_rows, unsigned int *counter, unsigned int *counter_next, int n_sms, cudaStream_t st)
{
    constexpr bool IS_INT = std::is_same<ACC, int>::value;
    constexpr bool IS_F32 = std::is_same<ACC, float>::value;
    const SlideSmem SM(sh.seg, sh.kc, sh.stages, sh.nsb, ROWS, IS_INT ? 4 : 8, PART, IS_F32, n_map_rows);
    auto kern = k_slide_bulk<T, ACC, ROWS, PART>;
    static std::atomic<int> smem_ok[64];                  // per instantiation (qld_allow_max_smem)
    cudaError_t e = qld_allow_max_smem(kern, smem_ok);
    if (e != cudaSuccess) return e;
    const int n_tiles = (int)((p.HW + SL_TP - 1) / SL_TP);
    cudaLaunchConfig_t lc;
    memset(&lc, 0, sizeof lc);
    lc.gridDim = dim3((unsigned)(n_tiles < n_sms ? n_tiles : n_sms));
    lc.blockDim = dim3(SL_THREADS);
    lc.dynamicSmemBytes = (size_t)SM.total + 128;
    lc.stream = st;
    // The three rotating tile counters are safe under the dependent launch only while launch w + 2 cannot start before launch w has
    // claimed its last tile (w + 2 zeroes the counter w counts on).  That holds when a CTA fills more than half of an SM's shared
    // memory -- then launch w + 1 becomes resident, and lets w + 2 go, only as the CTAs of w exit, and a CTA exits after its last
    // claim -- and when no tile is claimed through the counter at all (n_tiles <= grid: every CTA owns the tile of its index).
    // Any other shape (small forced tiles) is launched in plain stream order.
    static std::atomic<int> smem_per_sm[64];
    int dev = 0, per_sm = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < 64) per_sm = smem_per_sm[dev].load(std::memory_order_relaxed);
    if (per_sm == 0 && cudaDeviceGetAttribute(&per_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev) == cudaSuccess && dev >= 0 && dev < 64)
        smem_per_sm[dev].store(per_sm, std::memory_order_relaxed);
    const bool overlap_ok = n_tiles <= (int)lc.gridDim.x || (per_sm > 0 && 2 * (lc.dynamicSmemBytes + 1024) > (size_t)per_sm);
    cudaLaunchAttribute at;
    at.id = cudaLaunchAttributeProgrammaticStreamSerialization;    // may overlap the tail of the launch before it (see the kernel)
    at.val.programmaticStreamSerializationAllowed = overlap_ok ? 1 : 0;
    lc.attrs = &at;
    lc.numAttrs = 1;
    return cudaLaunchKernelEx(&lc, kern, *reinterpret_cast<const CUtensorMap *>(tmap), p, sh, n_map_rows, counter, counter_next);
}

template <typename T, typename ACC>
cudaError_t launch_slide_r(int rows, const void *tmap, const DemodParams &p, const SlideShape &sh, int n_map_rows, unsigned int *counter, unsigned int *counter_next, int n_sms, cudaStream_t st)
{
    const bool part = p.part != nullptr;
    switch (rows) {
    case 2: return part ? launch_slide_n<T, ACC, 2, true>(tmap, p, sh, n_map_rows, counter, counter_next, n_sms, st) : launch_slide_n<T, ACC, 2, false>(tmap, p, sh, n_map_rows, counter, counter_next, n_sms, st);
    case 3: return part ? launch_slide_n<T, ACC, 3, true>(tmap, p, sh, n_map_rows, counter, counter_next, n_sms, st) : launch_slide_n<T, ACC, 3, false>(tmap, p, sh, n_map_rows, counter, counter_next, n_sms, st);
    case 4: return part ? launch_slide_n<T, ACC, 4, true>(tmap, p, sh, n_map_rows, counter, counter_next, n_sms, st) : launch_slide_n<T, ACC, 4, false>(tmap, p, sh, n_map_rows, counter, counter_next, n_sms, st);
    default: return cudaErrorInvalidValue;
    }
}

int count_map_rows(const DemodParams &p) { return p.fin.K * ((p.fin.I != nullptr) + (p.fin.Q != nullptr) + (p.fin.amp != nullptr) + (p.fin.phase != nullptr)); }

}  // namespace

// Shape for this (dtype, rows, frame size), or seg = 0 when the kernel does not apply: rows beyond 4, a row pitch or base that
// is not 16-byte aligned, a frame too small to give every SM a tile (unless forced), or state buffers that leave no room for
// two frame stages.  force: 0 automatic, 1 use it whatever the frame size, 2 never.
SlideShape qld_slide_shape(int dtype, int kind, int rows, int part, int n_map_rows, int64_t HW, const void *frames, int n_sms, int force)
{
    SlideShape sh = {0, 0, 0, 0};
    if (force == 2 || rows > 4) return sh;
    const int bytes = dtype == QLD_U8 ? 1 : 2;
    if ((HW * bytes) % 16 != 0 || (reinterpret_cast<uintptr_t>(frames) & 15) != 0) return sh;
    const int64_t n_tiles = (HW + SL_TP - 1) / SL_TP;
    if (force != 1 && n_tiles < n_sms) return sh;
    const int seg = SL_TP * bytes;
    const int budget = 226 * 1024;
    // 16-frame stages with three state buffers when they fit; a large state (two references, partial sums, every map) leaves
    // room for two buffers and shorter stages only
    for (int kc = 16; kc >= 8; kc /= 2)
        for (int nsb = 3; nsb >= 2; --nsb) {
            const SlideSmem one(seg, kc, 1, nsb, rows, kind == 1 ? 4 : 8, part != 0, kind == 0, n_map_rows);
            const int fixed = nsb * one.state_bytes + 512;
            int stages = (budget - fixed) / (one.data_stage + one.w_stage);
            if (stages > 12) stages = 12;
            if (stages >= (nsb == 3 ? 3 : 2)) {
                sh.seg = seg; sh.kc = kc; sh.stages = stages; sh.nsb = nsb;
                return sh;
            }
        }
    return sh;
}

// 2-D tensor map over the frame store viewed as [cap frames][row_bytes / 8] 8-byte elements, box {seg / 8, kc}.
cudaError_t qld_slide_encode_tmap(void *tmap_out, const void *frames, int64_t row_bytes, int cap, const SlideShape &sh)
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

cudaError_t qld_launch_slide_bulk(int dtype, int kind, int rows, const void *tmap, const DemodParams &p, const SlideShape &sh,
                                  unsigned int *counter, unsigned int *counter_next, int n_sms, cudaStream_t st)
{
    const int n_map_rows = count_map_rows(p);
    const bool u8 = dtype == QLD_U8;
    switch (kind) {
    case 0: return u8 ? launch_slide_r<uint8_t, float>(rows, tmap, p, sh, n_map_rows, counter, counter_next, n_sms, st)
                      : launch_slide_r<uint16_t, float>(rows, tmap, p, sh, n_map_rows, counter, counter_next, n_sms, st);
    case 1: return u8 ? launch_slide_r<uint8_t, int>(rows, tmap, p, sh, n_map_rows, counter, counter_next, n_sms, st)
                      : launch_slide_r<uint16_t, int>(rows, tmap, p, sh, n_map_rows, counter, counter_next, n_sms, st);
    case 2: return u8 ? launch_slide_r<uint8_t, long long>(rows, tmap, p, sh, n_map_rows, counter, counter_next, n_sms, st)
                      : launch_slide_r<uint16_t, long long>(rows, tmap, p, sh, n_map_rows, counter, counter_next, n_sms, st);
    default: return cudaErrorInvalidValue;
    }
}

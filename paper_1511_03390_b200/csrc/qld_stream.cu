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
// stage.  Slices are combined through shared memory at the end of the tile (fp64 / int32), then the A4 epilogue
// runs with consecutive threads on consecutive pixels (coalesced accumulator and map traffic).  Variants with at
// most 32 accumulators per thread carry four more warps (10..13) that do nothing but this epilogue, out of a double
// buffered combine buffer, so that A4 of tile i overlaps the frame loop of tile i + 1 (hand-off by mbarriers:
// tile_known -> red_full -> red_empty).
//
// The frames of a launch are a list of runs (DemodRun): a whole window is one or two runs of weight +w, and the
// sliding update of PAPER.md:181-183 (A5) is the same kernel over {expired frames, -w} + {new frames, +w} with the
// sums added to the accumulators the previous window left in global memory.
#include "qld_device.cuh"
#include "qld_ptx.cuh"
#include "qld_stream.h"

using namespace qld_dev;
using namespace qld_ptx;

namespace {

constexpr int NW = 8;                 // consumer warps
// variants with at most 32 accumulators per thread get dedicated epilogue warps: A4 of tile i then overlaps the
// frame loop of tile i + 1, which pays when a launch has few frames per pixel (sliding updates, short windows)
// pixels per thread: at most QLD_STREAM_VB bytes of every frame.  16 (LDS.128) is the measured optimum: with 8 the
// eight consumer warps of a 2 KB segment own eight distinct column groups (TS = 1, no slices to combine, every
// thread finalises its own pixels from registers), but the per-frame overhead (weight loads, the one-hot branch) is
// then spread over half as many pixels: cfg3 hop 41 -> 46 us, integer whole window 196 -> 272 us.
#ifndef QLD_STREAM_VB
#define QLD_STREAM_VB 16
#endif
constexpr int stream_v(int bytes, int rows)
{
    int v = qld_dev::pick_v(bytes, rows);
    const int cap = QLD_STREAM_VB / bytes;
    if (v > cap) v = cap;
    // prefer 32 accumulators (128 registers, room for the epilogue warps) as long as a thread keeps 8 bytes per frame
    while (rows * v > 32 && v * bytes > 8) v /= 2;
    return v;
}
constexpr bool stream_light(int bytes, int rows) { return rows * stream_v(bytes, rows) <= 32; }
// four epilogue warps for the variants whose frame loop fits in 128 registers (13 warps per CTA)
constexpr int stream_nepi(int bytes, int rows) { return stream_light(bytes, rows) ? 4 : 0; }
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
        total = off_bar + 2 * stages * 8 + TQ * 4 + 6 * 8 + 16;
    }
};

// PART: block-partial sliding (8(f3)): the launch's sums are also stored in p.part (after the slot's old content was
// taken off the stored sums when p.part_sub is set)
template <typename T, typename ACC, int ROWS, int V, int NWT, int NEPI, bool PART>
__global__ void __launch_bounds__(32 * (NWT + 1 + NEPI), 1)
k_demod_stream(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ DemodParams p, const StreamShape sh, unsigned int *tile_counter,
               unsigned int *counter_next)
{
    using PX = Pix<T, V>;
    constexpr bool IS_INT = std::is_same<ACC, int>::value;
    using RED = typename std::conditional<IS_INT, int, double>::type;
    constexpr int VB = V * (int)sizeof(T);                 // bytes per thread per frame

    const int SEG = sh.seg, KC = sh.kc, STAGES = sh.stages;
    const int CG = SEG / (32 * VB), TS = NWT / CG;          // column groups, time slices
    // combine buffer: [ROWS (+1: pedestal)][V][RS] RED cells, RS = column count padded so that the epilogue's
    // pixel-order reads (v fastest) fall into distinct banks
    constexpr int PAD = 128 / ((int)sizeof(RED) * V) > 0 ? 128 / ((int)sizeof(RED) * V) : 1;
    constexpr int RROWS = ROWS + (IS_INT ? 0 : 1);
    // pixels per thread whose stored sums are prefetched in a sliding update (about 32 registers)
    constexpr int PFN_ = (IS_INT ? 32 : 16) / ROWS;
    constexpr int PFN = PFN_ >= 8 ? 8 : (PFN_ >= 4 ? 4 : (PFN_ >= 2 ? 2 : 1));      // a power of two (batches of four)
    const int RS = CG * 32 + PAD;
    // epilogue warps (NEPI > 0): the combine buffer is double buffered and finalised by them
    const bool SPLIT = NEPI > 0 && TS > 1;
    const int red_cells = RROWS * V * RS;
    const StreamSmem SM(SEG, KC, STAGES, ROWS, TS > 1 ? (SPLIT ? 2 : 1) * red_cells * (int)sizeof(RED) : 0);

    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    unsigned char *sData = smem;
    ACC *sW = reinterpret_cast<ACC *>(smem + SM.off_w);
    RED *red = reinterpret_cast<RED *>(smem + SM.off_red);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + SM.off_bar);
    uint64_t *empty = full + STAGES;
    volatile int *tile_q = reinterpret_cast<volatile int *>(empty + STAGES);
    uint64_t *red_full = reinterpret_cast<uint64_t *>(const_cast<int *>(tile_q) + TQ);   // [2] consumers -> epilogue warps
    uint64_t *red_empty = red_full + 2, *tile_known = red_full + 4;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t row_bytes = p.HW * (int64_t)sizeof(T);
    const int n_tiles = (int)((row_bytes + SEG - 1) / SEG);

    if (threadIdx.x == 0) {
        if (blockIdx.x == 0) *counter_next = 0;   // the next launch's tile counter (the two alternate: no memset between launches)
        for (int i = 0; i < STAGES; ++i) {
            mbar_init(&full[i], 2);          // the producer's expect_tx arrival + its "weights written" arrival
            mbar_init(&empty[i], NWT);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(&red_full[i], NWT * 32);
            mbar_init(&red_empty[i], NEPI > 0 ? NEPI * 32 : 1);
            mbar_init(&tile_known[i], 1);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == 0) {
        // ===== producer: TMA boxes + weight rows, tile scheduler =====
        const ACC *wtab = static_cast<const ACC *>(p.wtab);
        int stage = 0, it = 0;
        uint32_t phase = 0;
        // the first tile of a CTA is its block index (no round trip before the first copy); later ones come from the
        // global counter, claimed one tile ahead so that the atomic's latency hides under the current tile's copies
        int next = (int)blockIdx.x;
        for (;; ++it) {
            int tile = 0;
            if (lane == 0) {
                tile = next < n_tiles ? next : -1;
                if (tile >= 0) next = (int)gridDim.x + (int)atomicAdd(tile_counter, 1u);
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
            for (int run = 0; run < p.n_runs; ++run) {
                const int rn = p.run[run].n, rslot = p.run[run].slot0, rw0 = p.run[run].w0;
                const ACC sgn = (ACC)p.run[run].sign;
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
                        int e = rw0 + c0 + i / ROWS;           // rw0 < cap_w and c0 + i / ROWS < cap_w
                        if (e >= p.cap_w) e -= p.cap_w;
                        wdst[i] = sgn * __ldg(wtab + (int64_t)e * ROWS + (i % ROWS));
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&full[stage]);
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
            }
        }
        return;
    }

    // ---- A4 for the pixels q0, q0 + qstride, ... of a tile whose combined sums sit in `redb` (consecutive threads on
    // consecutive pixels: coalesced accumulator and map traffic).  prefetch_acc requests, ahead of time, the previous
    // window's sums (A5) of the same pixels.
    const int TP = SEG / (int)sizeof(T);                   // pixels per tile
    auto prefetch_acc = [&](int tile, int q0, int qstride, RED (&pf)[PFN][ROWS]) {
        const RED *accg = static_cast<const RED *>(p.acc_out);
        const int64_t tile_pix0 = (int64_t)tile * TP;
#pragma unroll
        for (int i = 0; i < PFN; ++i) {
            const int q = q0 + i * qstride;
            const bool ok = q < TP && tile_pix0 + q < p.HW;
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                pf[i][r] = ok ? accg[(int64_t)r * p.HW + tile_pix0 + q] : (RED)0;
                if constexpr (PART) {
                    if (p.part_sub && ok) pf[i][r] -= static_cast<const RED *>(p.part)[(int64_t)r * p.HW + tile_pix0 + q];
                }
            }
        }
    };
    auto finalise_tile = [&](const RED *redb, int tile, int q0, int qstride, const RED (&pf)[PFN][ROWS], bool use_pf) {
        const int64_t tile_pix0 = (int64_t)tile * TP;
        RowVals<double, ROWS> wsum;
#pragma unroll
        for (int r = 0; r < ROWS; ++r) wsum.a[r] = 0.0;
        if constexpr (!IS_INT) {
#pragma unroll
            for (int r = 0; r < ROWS; ++r) wsum.a[r] = p.cum[(int64_t)p.cum_hi * ROWS + r] - p.cum[(int64_t)p.cum_lo * ROWS + r];
        }
        auto finalise_q = [&](int q, int64_t pixel, const RED *prev) {
            const int v = q % V, tc = q / V;
            RED *accg = static_cast<RED *>(p.acc_out);
            double ped = 0.0;
            if constexpr (!IS_INT) ped = redb[(size_t)(ROWS * V + v) * RS + tc];
            RowVals<RED, ROWS> a;
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                a.a[r] = redb[(size_t)(r * V + v) * RS + tc];
                RED old = 0;
                if constexpr (PART) {                      // 8(f3): this launch's sums replace the expired batch's
                    RED *partg = static_cast<RED *>(p.part);
                    if (p.part_sub && !prev) old = partg[(int64_t)r * p.HW + pixel];
                    partg[(int64_t)r * p.HW + pixel] = a.a[r];
                }
                if (p.acc_add) a.a[r] += prev ? prev[r] : accg[(int64_t)r * p.HW + pixel] - old;
                if (accg) accg[(int64_t)r * p.HW + pixel] = a.a[r];
            }
            if constexpr (!IS_INT) {
                if (p.ped_out) p.ped_out[pixel] = (float)ped;
            }
            finalise_pixel_nl<ROWS, IS_INT, RED>(&p.fin, a, ped, wsum, pixel, p.HW);   // sum x w = sum (x - ped) w + ped * sum w
        };
        if (use_pf && p.fin.K == 1) {
            // one reference, stored sums prefetched: the pixels of a thread go through the fp64 arithmetic in batches of
            // four with no branch between them (independent dependency chains interleave), stores predicated at the end
            constexpr int B = PFN < 4 ? PFN : 4;
            const FinParams &f = p.fin;
            RED *accg = static_cast<RED *>(p.acc_out);
#pragma unroll
            for (int i0 = 0; i0 < PFN; i0 += B) {
                RED a[B][ROWS];
                double S[B], C[B], pedv[B];
                bool ok[B];
                int64_t pix[B];
#pragma unroll
                for (int j = 0; j < B; ++j) {
                    const int q = q0 + (i0 + j) * qstride;
                    ok[j] = q < TP && tile_pix0 + q < p.HW;
                    const int qq = ok[j] ? q : q0;
                    pix[j] = tile_pix0 + qq;
                    const int v = qq % V, tc = qq / V;
                    pedv[j] = 0.0;
                    if constexpr (!IS_INT) pedv[j] = redb[(size_t)(ROWS * V + v) * RS + tc];
#pragma unroll
                    for (int r = 0; r < ROWS; ++r) {
                        a[j][r] = redb[(size_t)(r * V + v) * RS + tc];
                        if constexpr (PART) {
                            if (ok[j]) static_cast<RED *>(p.part)[(int64_t)r * p.HW + pix[j]] = a[j][r];
                        }
                        if (p.acc_add) a[j][r] += pf[i0 + j][r];
                    }
                }
#pragma unroll
                for (int j = 0; j < B; ++j) {
                    if constexpr (IS_INT) {
                        S[j] = 0.0; C[j] = 0.0;
#pragma unroll
                        for (int r = 0; r < ROWS; ++r) {
                            const double x = (double)a[j][r];
                            S[j] = fma(x, f.sw[r], S[j]);
                            C[j] = fma(x, f.cw[r], C[j]);
                        }
                    } else {
                        S[j] = (double)a[j][0] + pedv[j] * wsum.a[0];       // sum x w = sum (x - ped) w + ped * sum w
                        C[j] = (double)a[j][1] + pedv[j] * wsum.a[1];
                    }
                    rotate_iq(f.rot, 0, S[j], C[j]);
                    S[j] *= f.scale;
                    C[j] *= f.scale;
                }
                float amp[B], ph[B];
#pragma unroll
                for (int j = 0; j < B; ++j) amp[j] = f.amp ? (float)sqrt(S[j] * S[j] + C[j] * C[j]) : 0.0f;
#pragma unroll
                for (int j = 0; j < B; ++j) ph[j] = (f.phase && !(S[j] == 0.0 && C[j] == 0.0)) ? (float)atan2(C[j], S[j]) : 0.0f;
#pragma unroll
                for (int j = 0; j < B; ++j) {
                    if (!ok[j]) continue;
                    if (accg) {
#pragma unroll
                        for (int r = 0; r < ROWS; ++r) accg[(int64_t)r * p.HW + pix[j]] = a[j][r];
                    }
                    if constexpr (!IS_INT) {
                        if (p.ped_out) p.ped_out[pix[j]] = (float)pedv[j];
                    }
                    if (f.I) f.I[pix[j]] = (float)S[j];
                    if (f.Q) f.Q[pix[j]] = (float)C[j];
                    if (f.amp) f.amp[pix[j]] = amp[j];
                    if (f.phase) f.phase[pix[j]] = ph[j];
                }
            }
        } else if (use_pf) {
#pragma unroll
            for (int i = 0; i < PFN; ++i) {
                const int q = q0 + i * qstride;
                if (q < TP && tile_pix0 + q < p.HW) finalise_q(q, tile_pix0 + q, pf[i]);
            }
        } else {
            for (int q = q0; q < TP; q += qstride) {
                if (tile_pix0 + q >= p.HW) break;
                finalise_q(q, tile_pix0 + q, nullptr);
            }
        }
    };

    if (warp > NWT) {
        // ===== epilogue warps: finalise tile i from red[i & 1] while the consumers run the frame loop of tile i + 1 =====
        if (!SPLIT) return;
        const int et = (warp - 1 - NWT) * 32 + lane;
        const bool use_pf = TP <= PFN * NEPI * 32;          // every pixel of the tile has a register slot
        for (int it = 0;; ++it) {
            const int buf = it & 1;
            const uint32_t par = (uint32_t)(it >> 1) & 1u;
            mbar_wait(&tile_known[buf], par);
            const int tile = tile_q[it & (TQ - 1)];
            if (tile < 0) break;
            RED pf[PFN][ROWS];
            if (use_pf && p.acc_add) prefetch_acc(tile, et, NEPI * 32, pf);
            mbar_wait(&red_full[buf], par);
            finalise_tile(red + (size_t)buf * red_cells, tile, et, NEPI * 32, pf, use_pf);
            mbar_arrive(&red_empty[buf]);
        }
        return;
    }

    // ===== consumers =====
    const uint32_t bsw = p.big_endian ? 0x11u : 0u;
    const int cw = warp - 1, cg = cw % CG, ts = cw / CG;
    const int col = (cg * 32 + lane) * VB;                 // byte offset of this thread's pixels inside the segment
    const int tcol = cg * 32 + lane;                       // thread column inside the tile
    int stage = 0;
    uint32_t phase = 0;
    for (int it = 0;; ++it) {
        mbar_wait(&full[stage], phase);
        const int tile = tile_q[it & (TQ - 1)];
        const int buf = SPLIT ? (it & 1) : 0;
        RED *redb = red + (size_t)buf * red_cells;
        if (SPLIT) {
            // red[buf] was last used by tile it - 2: wait until the epilogue warps are done with it, then tell them which
            // tile comes next in this buffer (they prefetch its stored sums while the frame loop runs)
            if (it >= 2) mbar_wait(&red_empty[buf], ((uint32_t)(it >> 1) & 1u) ^ 1u);
            if (cw == 0 && lane == 0) mbar_arrive(&tile_known[buf]);
        }
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
        bool need_ped = !IS_INT;
        if constexpr (!IS_INT) {
            if (p.ped_in != nullptr) {                     // A5: the pedestal the accumulators were seeded with
                need_ped = false;
                if (active) {
#pragma unroll
                    for (int v = 0; v < V; ++v) pedm[v] = 8388608.0f + __ldg(p.ped_in + pix0 + v);
                }
            }
        }

        // without epilogue warps the consumers finalise: request the stored sums now, under the frame loop
        RED pf[PFN][ROWS];
        const bool use_pf = !SPLIT && TS > 1 && TP <= PFN * NWT * 32;
        if (use_pf && p.acc_add) prefetch_acc(tile, cw * 32 + lane, NWT * 32, pf);

        // one slice per column group: the thread finalises its own V pixels; their stored sums (A5) are requested now
        // (a 2 KB segment has eight column groups only when a thread takes at most 8 bytes per frame)
        constexpr bool CAN_OWN = VB <= 8;
        // (prefetched only where that costs at most 32 registers; the 64-accumulator variants load them in the epilogue)
        constexpr bool OWN_PF = CAN_OWN && ROWS * V * (int)sizeof(RED) <= 128;
        RED prev[OWN_PF ? ROWS : 1][OWN_PF ? V : 1];
        const bool own_prev = CAN_OWN && TS == 1 && p.acc_add && active;
        if constexpr (OWN_PF) {
            if (own_prev) {
                const RED *accg = static_cast<const RED *>(p.acc_out);
#pragma unroll
                for (int r = 0; r < ROWS; ++r) {
                    load_vec<RED, V>(accg + (int64_t)r * p.HW + pix0, prev[r]);
                    if (PART && p.part_sub) {
                        RED old[V];
                        load_vec<RED, V>(static_cast<const RED *>(p.part) + (int64_t)r * p.HW + pix0, old);
#pragma unroll
                        for (int v = 0; v < V; ++v) prev[r][v] -= old[v];
                    }
                }
            }
        }

        bool first = true;
        for (int run = 0; run < p.n_runs; ++run) {
            const int rn = p.run[run].n;
            for (int c0 = 0; c0 < rn; c0 += KC) {
                const int nf = min(KC, rn - c0);
                if (!first) mbar_wait(&full[stage], phase);
                const unsigned char *d = sData + (size_t)stage * SM.data_stage + col;
                const ACC *wrow = sW + (size_t)stage * KC * ROWS;
                if (first) {
                    first = false;
                    if (need_ped) {
                        // pedestal = the pixel's first sample in the window (exact integer), DESIGN.md "Precision"
                        uint32_t w0[PX::NW];
                        PX::load_shared(d, w0);
#pragma unroll
                        for (int v = 0; v < V; ++v) pedm[v] = PX::getf_biased(w0, v, bsw);
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
                        for (int u = 0; u < 4; ++u) {
                            if constexpr (IS_INT) {
                                if (p.onehot) { accumulate_onehot<T, ROWS, V>(w[u], wt[u], acc, bsw); continue; }
                            }
                            accumulate<T, ACC, ROWS, V>(w[u], wt[u], pedm, acc, bsw);
                        }
                    }
                } else {
                    for (; f < nf; f += TS) {
                        uint32_t w[PX::NW];
                        ACC wt[ROWS];
                        PX::load_shared(d + (size_t)f * SEG, w);
                        load_weights_shared<ACC, ROWS>(wrow + f * ROWS, wt);
                        if constexpr (IS_INT) {
                            if (p.onehot) { accumulate_onehot<T, ROWS, V>(w, wt, acc, bsw); continue; }
                        }
                        accumulate<T, ACC, ROWS, V>(w, wt, pedm, acc, bsw);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[stage]);
                if (++stage == STAGES) { stage = 0; phase ^= 1; }
            }
        }

        if (TS > 1) {
            // ---- combine the TS time slices (fp64 / int32).  The ROWS*V values of a thread are cut into NWT chunks;
            // in turn j slice ts adds the chunks c with c = ts + j (mod TS), so every slice works in every turn and
            // no two slices touch a cell in the same turn.  Turn 0 stores (first touch), later turns add.
            constexpr int CH = ROWS * V / NWT;
            static_assert(CH >= 1 && CH * NWT == ROWS * V, "chunking");
            for (int j = 0; j < TS; ++j) {
                const int want = (ts + j) & (TS - 1);
#pragma unroll
                for (int c = 0; c < NWT; ++c) {
                    if ((c & (TS - 1)) != want) continue;
                    RED t[CH];
#pragma unroll
                    for (int e = 0; e < CH; ++e) {
                        const int i = c * CH + e;
                        t[e] = (j == 0) ? (RED)0 : redb[(size_t)i * RS + tcol];
                    }
#pragma unroll
                    for (int e = 0; e < CH; ++e) {
                        const int i = c * CH + e;
                        redb[(size_t)i * RS + tcol] = t[e] + (RED)acc[i / V][i % V];
                    }
                }
                if constexpr (!IS_INT) {
                    if (j == 0 && ts == 0) {
#pragma unroll
                        for (int v = 0; v < V; ++v) redb[(size_t)(ROWS * V + v) * RS + tcol] = (RED)(pedm[v] - 8388608.0f);
                    }
                }
                if (SPLIT && j == TS - 1) mbar_arrive(&red_full[buf]);   // every consumer thread: its cells are written
                else named_barrier(1, NWT * 32);
            }
            if (!SPLIT) {
                finalise_tile(redb, tile, cw * 32 + lane, NWT * 32, pf, use_pf);
                named_barrier(1, NWT * 32);                 // red is free for the next tile
            }
        } else if (CAN_OWN && active) {
          if constexpr (CAN_OWN) {
            // one slice per column group: every thread finalises its own V pixels from registers, 16-byte accesses
            RED *accg = static_cast<RED *>(p.acc_out);
            RED a[ROWS][V];
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
#pragma unroll
                for (int v = 0; v < V; ++v) a[r][v] = (RED)acc[r][v];
                if constexpr (PART) {
                    RED *partg = static_cast<RED *>(p.part) + (int64_t)r * p.HW + pix0;
                    RED old[V];
#pragma unroll
                    for (int v = 0; v < V; ++v) old[v] = 0;
                    if (!OWN_PF && p.part_sub) load_vec<RED, V>(partg, old);
                    store_vec<RED, V>(partg, a[r]);
#pragma unroll
                    for (int v = 0; v < V; ++v) a[r][v] -= old[v];
                }
                if constexpr (OWN_PF) {
#pragma unroll
                    for (int v = 0; v < V; ++v) a[r][v] += (own_prev ? prev[r][v] : (RED)0);
                } else if (own_prev) {
                    RED t[V];
                    load_vec<RED, V>(accg + (int64_t)r * p.HW + pix0, t);
#pragma unroll
                    for (int v = 0; v < V; ++v) a[r][v] += t[v];
                }
                if (accg) store_vec<RED, V>(accg + (int64_t)r * p.HW + pix0, a[r]);
            }
            float pedf[V];
#pragma unroll
            for (int v = 0; v < V; ++v) pedf[v] = pedm[v] - 8388608.0f;
            if constexpr (!IS_INT) {
                if (p.ped_out) store_vec<float, V>(p.ped_out + pix0, pedf);
            }
            const FinParams &f = p.fin;
            for (int k = 0; k < f.K; ++k) {
                float oI[V], oQ[V], oA[V], oP[V];
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
                    } else {
#pragma unroll
                        for (int r = 0; r + 1 < ROWS; r += 2)
                            if (r == 2 * k) {
                                const double ws = p.cum[(int64_t)p.cum_hi * ROWS + r] - p.cum[(int64_t)p.cum_lo * ROWS + r];
                                const double wc = p.cum[(int64_t)p.cum_hi * ROWS + r + 1] - p.cum[(int64_t)p.cum_lo * ROWS + r + 1];
                                S = (double)a[r][v] + (double)pedf[v] * ws;          // sum x w = sum (x - ped) w + ped * sum w
                                C = (double)a[r + 1][v] + (double)pedf[v] * wc;
                            }
                    }
                    rotate_iq(f.rot, k, S, C);
                    S *= f.scale;
                    C *= f.scale;
                    oI[v] = (float)S;
                    oQ[v] = (float)C;
                    oA[v] = f.amp ? (float)sqrt(S * S + C * C) : 0.0f;
                    oP[v] = (f.phase && !(S == 0.0 && C == 0.0)) ? (float)atan2(C, S) : 0.0f;
                }
                const int64_t o = (int64_t)k * p.HW + pix0;
                if (f.I) store_vec<float, V>(f.I + o, oI);
                if (f.Q) store_vec<float, V>(f.Q + o, oQ);
                if (f.amp) store_vec<float, V>(f.amp + o, oA);
                if (f.phase) store_vec<float, V>(f.phase + o, oP);
            }
          }
        }
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int red_bytes_for(int seg, int vb, int rows, int v, bool is_int, int nw, int nepi)
{
    const int cg = seg / (32 * vb), ts = nw / cg;
    const int esz = is_int ? 4 : 8;
    const int pad = 128 / (esz * v) > 0 ? 128 / (esz * v) : 1;
    return ts > 1 ? (nepi > 0 ? 2 : 1) * (rows + (is_int ? 0 : 1)) * v * (cg * 32 + pad) * esz : 0;
}

template <typename T, typename ACC, int ROWS, int NWT, int NEPI, bool PART>
cudaError_t launch_stream_n(const void *tmap, const DemodParams &p, const StreamShape &sh, unsigned int *counter, unsigned int *counter_next, int n_sms, cudaStream_t st)
{
    constexpr int V = stream_v(sizeof(T), ROWS);
    constexpr bool IS_INT = std::is_same<ACC, int>::value;
    const StreamSmem SM(sh.seg, sh.kc, sh.stages, ROWS, red_bytes_for(sh.seg, V * (int)sizeof(T), ROWS, V, IS_INT, NWT, NEPI));
    auto kern = k_demod_stream<T, ACC, ROWS, V, NWT, NEPI, PART>;
    static std::atomic<int> smem_ok[64];                  // per instantiation (qld_allow_max_smem)
    cudaError_t e = qld_allow_max_smem(kern, smem_ok);
    if (e != cudaSuccess) return e;
    const int64_t row_bytes = p.HW * (int64_t)sizeof(T);
    const int n_tiles = (int)((row_bytes + sh.seg - 1) / sh.seg);
    kern<<<n_tiles < n_sms ? n_tiles : n_sms, 32 * (NWT + 1 + NEPI), SM.total + 128, st>>>(*reinterpret_cast<const CUtensorMap *>(tmap), p, sh, counter, counter_next);
    return cudaGetLastError();
}

template <typename T, typename ACC, int ROWS>
cudaError_t launch_stream_t(const void *tmap, const DemodParams &p, const StreamShape &sh, unsigned int *counter, unsigned int *counter_next, int n_sms, cudaStream_t st)
{
    if (p.part) return launch_stream_n<T, ACC, ROWS, NW, stream_nepi(sizeof(T), ROWS), true>(tmap, p, sh, counter, counter_next, n_sms, st);
    return launch_stream_n<T, ACC, ROWS, NW, stream_nepi(sizeof(T), ROWS), false>(tmap, p, sh, counter, counter_next, n_sms, st);
}

template <typename T, typename ACC>
cudaError_t launch_stream_r(int rows, const void *tmap, const DemodParams &p, const StreamShape &sh, unsigned int *counter, unsigned int *counter_next, int n_sms, cudaStream_t st)
{
    switch (rows) {
    case 2: return launch_stream_t<T, ACC, 2>(tmap, p, sh, counter, counter_next, n_sms, st);
    case 3: return launch_stream_t<T, ACC, 3>(tmap, p, sh, counter, counter_next, n_sms, st);
    case 4: return launch_stream_t<T, ACC, 4>(tmap, p, sh, counter, counter_next, n_sms, st);
    case 8: return launch_stream_t<T, ACC, 8>(tmap, p, sh, counter, counter_next, n_sms, st);
    case 16: return launch_stream_t<T, ACC, 16>(tmap, p, sh, counter, counter_next, n_sms, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace

// Tile shape for this (dtype, rows, frame size), or seg = 0 when the streaming kernel does not apply (row pitch or
// base not 16-byte aligned, or a frame too small to give every SM a tile: k_demod_whole handles those).
StreamShape qld_stream_shape(int dtype, int is_int, int rows, int64_t HW, const void *frames, int n_sms, int force_seg, int force_kc)
{
    StreamShape sh = {0, 0, 0};
    const int bytes = dtype == QLD_U8 ? 1 : 2;
    const int v = stream_v(bytes, rows), vb = v * bytes;
    const int64_t row_bytes = HW * bytes;
    if (row_bytes % 16 != 0 || (reinterpret_cast<uintptr_t>(frames) & 15) != 0) return sh;
    const int nw = NW;
    int seg = 2048;                                        // TMA box: at most 256 8-byte elements per row
    if (seg > nw * 32 * vb) seg = nw * 32 * vb;
    // small frames: at least two tiles per SM, but segments as wide as that allows (cfg1 sweep: 1 KB x 32 frames
    // 41 us, 512 B x 32 frames 47 us: narrow rows cost more per byte and need more time slices to combine)
    while (seg > 32 * vb && (row_bytes + seg - 1) / seg < 2 * (int64_t)n_sms) seg /= 2;
    int kc = 32768 / seg > 16 ? 32768 / seg : 16, stages = 0;      // stages of at least 32 KB
    bool forced = false;
    if (force_seg > 0) {                                   // debug / test override (qld_debug_set_tile)
        const int s2 = force_seg, k2 = force_kc;
        if (s2 >= 32 * vb && s2 <= nw * 32 * vb && s2 <= 2048 && (s2 & (s2 - 1)) == 0 && k2 >= 4 && k2 <= 256) { seg = s2; kc = k2; forced = true; }
    }
    if (!forced && (row_bytes + seg - 1) / seg < n_sms) return sh;
    const int ts = nw / (seg / (32 * vb));
    if (kc < 4 * ts) kc = 4 * ts;                          // every slice gets a multiple of four frames per stage
    kc = (kc + 4 * ts - 1) / (4 * ts) * (4 * ts);
    const int red = red_bytes_for(seg, vb, rows, v, is_int != 0, nw, stream_nepi(bytes, rows));
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
                                    unsigned int *counter, unsigned int *counter_next, int n_sms, cudaStream_t st)
{
    if (dtype == QLD_U8)
        return is_int ? launch_stream_r<uint8_t, int>(rows, tmap, p, sh, counter, counter_next, n_sms, st) : launch_stream_r<uint8_t, float>(rows, tmap, p, sh, counter, counter_next, n_sms, st);
    return is_int ? launch_stream_r<uint16_t, int>(rows, tmap, p, sh, counter, counter_next, n_sms, st) : launch_stream_r<uint16_t, float>(rows, tmap, p, sh, counter, counter_next, n_sms, st);
}

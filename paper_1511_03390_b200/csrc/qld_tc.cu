// Tensor-core demodulation (SURVEY.md 8(a) rows A3 / A6 on tcgen05): the window sum
//     row_r(p) = sum_s x_s(p) * R_r(s)          (R_r = fixed-point reference, Q1.30 integers)
// as the contraction [pixel-bytes x frames] . [frames x digits] on the 5th-generation tensor cores, exact in
// integers (kind::i8, int32 accumulators in TMEM).
//
// Why this shape.  The frame stack is frame-major, so for a fixed frame the bytes of adjacent pixels are
// contiguous: the A operand [M = pixel bytes][K = frames] is "MN-major" and TMA boxes of {128 bytes, 8 frames}
// with 128-byte swizzle land in shared memory in exactly the canonical layout tcgen05.mma reads -- the raw
// camera bytes go global -> shared -> tensor core with no conversion pass and no CUDA-core instruction per
// sample.  A uint16 sample x = lo + 256*hi occupies two M rows (its two little-endian bytes); a reference
// R = sum_j d_j 256^j is split into four signed base-256 digits d_j in [-128, 127] (four N columns).  The MMA
// produces P[byte][j] = sum_s byte_s * d_j(s) (|P| <= 255*128*N, exact in int32) and the epilogue recombines
//     sum_s x_s R_s = sum_b sum_j 256^(b+j) P[b][j]     exactly in int64.
// The kernel is HBM-bound for any K <= 8 (N columns = 8K <= 64): per 32-frame MMA step the tensor pipe needs
// 128*N/256 <= 32 cycles for 4 KB of samples, about five times faster than HBM delivers them to one SM.
//
// Structure (one persistent CTA per SM, 192 threads): warp 0 = TMA producer, warp 1 = MMA issuer, warps 2-5 =
// epilogue (TMEM -> registers -> maps).  A CTA tile is T adjacent 128-byte pixel spans over all frames; the
// accumulators of a tile (T * NC columns) are double buffered in TMEM so the epilogue of tile i overlaps the
// main loop of tile i+1.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "qld_angle.cuh"
#include "qld_internal.h"
#include "qld_ptx.cuh"
#include "qld_tc.h"

using namespace qld_ptx;
using qld_angle::half_turns_of;

namespace {

constexpr int KC_PAD = 64;        // the digit tiles are padded to a multiple of this many frames
constexpr int SUB_BYTES = 128;    // pixel bytes per MMA M tile
constexpr int MMA_K = 32;         // frames per tcgen05.mma (8-bit operands)
constexpr int GRP = 8;            // frames per 128-byte-swizzle atom (8 rows of 128 bytes = 1 KB)
constexpr int TC_TQ = 16;         // tile-id queue entries: the producer runs at most `stages` <= 12 tiles ahead of the MMA warp
constexpr int TC_MAX_STAGES = 12;
static_assert(TC_MAX_STAGES < TC_TQ, "the tile queue must outlast the producer's run-ahead");

// ---------------------------------------------------------------------------------------------------
// PTX wrappers
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tc_mma_i8(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tc_ld16(uint32_t taddr, uint32_t (&r)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                   "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr));
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// shared-memory matrix descriptor (cute::UMMA::SmemDescriptor bit layout): start address, leading and stride
// byte offsets in 16-byte units, version 1 (Blackwell), layout type in bits [61,64)
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes, uint32_t layout_type)
{
    return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16) | ((uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32) |
           (1ull << 46) | ((uint64_t)layout_type << 61);
}

// ---------------------------------------------------------------------------------------------------
// fixed-point reference table and its digit tiles
// ---------------------------------------------------------------------------------------------------
// rfix[r][s-1] = rint(2^30 * sin or cos(theta_{k,s})), r = 2k (sin) / 2k+1 (cos), s = 1..n
__global__ void k_fixed_table_fill(TableFillParams p, int32_t *rfix, int n_stride)
{
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < p.n * p.K; idx += gridDim.x * blockDim.x) {
        const int i = idx / p.K, k = idx % p.K;
        double sn, cs;
        sincospi(half_turns_of(p.ref[k], p.s_first + i), &sn, &cs);
        rfix[(int64_t)(2 * k) * n_stride + i] = (int32_t)rint(sn * 1073741824.0);
        rfix[(int64_t)(2 * k + 1) * n_stride + i] = (int32_t)rint(cs * 1073741824.0);
    }
}

__global__ void k_fixed_from_doubles(const double *tab, int n, int k, int32_t *rfix, int n_stride)
{
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        rfix[(int64_t)(2 * k) * n_stride + i] = (int32_t)rint(tab[i] * 1073741824.0);
        rfix[(int64_t)(2 * k + 1) * n_stride + i] = (int32_t)rint(tab[n + i] * 1073741824.0);
    }
}

// digit tiles: for MMA step q (32 frames) a block of NC*32 bytes laid out [n/8][k/16][n%8][k%16] (the
// no-swizzle K-major canonical layout: 8x16-byte core matrices, LBO = 128 B between K halves, SBO = 256 B
// between groups of 8 columns).  Column c = 4*r + j holds digit j of reference row r.
__global__ void k_digit_pack(const int32_t *rfix, int n_stride, int n, int rows, int nc, int n_steps, int8_t *digits)
{
    const int64_t total = (int64_t)n_steps * nc * MMA_K;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int q = (int)(idx / (nc * MMA_K));
        const int rem = (int)(idx % (nc * MMA_K));
        const int k0 = rem & 15, n0 = (rem >> 4) & 7, k1 = (rem >> 7) & 1, n1 = rem >> 8;
        const int c = n1 * 8 + n0, kk = k1 * 16 + k0;
        const int s = q * MMA_K + kk, r = c >> 2, j = c & 3;
        int d = 0;
        if (s < n && r < rows) {
            int32_t v = rfix[(int64_t)r * n_stride + s];
            for (int t = 0; t <= j; ++t) {
                d = ((v + 128) & 255) - 128;      // balanced digit in [-128, 127]
                v = (v - d) >> 8;                 // exact: v - d is a multiple of 256
            }
        }
        digits[idx] = (int8_t)d;
    }
}

// ---------------------------------------------------------------------------------------------------
// the contraction kernel
// ---------------------------------------------------------------------------------------------------
// shared-memory carve-up for (NC columns, T spans per tile, STAGES pipeline stages)
struct TcSmem {
    int a_stage, b_stage, off_b, off_bar, total;
    __host__ __device__ TcSmem(int nc, int t, int stages, int kc)
    {
        a_stage = t * kc * SUB_BYTES;                 // [kc/8 frame groups][t spans][8 frames][128 bytes]
        b_stage = (kc / MMA_K) * nc * MMA_K;
        off_b = stages * a_stage;
        off_bar = off_b + stages * b_stage;
        total = off_bar + (2 * stages + 4) * 8 + 16 + 8 + TC_TQ * 4 + 8;   // barriers, TMEM slot, tile queue, tbuf_tile
    }
};

template <int NC, int BYTES>
__global__ void __launch_bounds__(192, 1) k_demod_tc(const __grid_constant__ CUtensorMap tmap2, const __grid_constant__ CUtensorMap tmap4,
                                                     const TcParams p, const int T, const int STAGES, const int KC, const int use4d)
{
    const TcSmem SM(NC, T, STAGES, KC);
    extern __shared__ unsigned char smem_raw[];
    // 128-byte-swizzled TMA/UMMA tiles need 1024-byte alignment in the shared window
    unsigned char *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    unsigned char *sA = smem;
    unsigned char *sB = smem + SM.off_b;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + SM.off_bar);
    uint64_t *empty = full + STAGES;
    uint64_t *tfull = empty + STAGES;
    uint64_t *tempty = tfull + 2;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tempty + 2);
    volatile int *tile_q = reinterpret_cast<volatile int *>(tmem_slot + 2);      // [TC_TQ] tile ids, producer -> MMA warp
    volatile int *tbuf_tile = tile_q + TC_TQ;                                        // [2] tile id per accumulator buffer

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_chunks = (p.N + KC - 1) / KC;
    const int n_full = p.N / GRP * GRP;               // frames covered by whole 8-frame groups (the 4-D map's extent)
    const int n_sub = (int)((p.row_bytes + SUB_BYTES - 1) / SUB_BYTES);
    const int n_tiles = (n_sub + T - 1) / T;

    if (threadIdx.x == 0) {
        for (int i = 0; i < STAGES; ++i) {
            mbar_init(&full[i], 1);
            mbar_init(&empty[i], 1);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(&tfull[i], 2);
            mbar_init(&tempty[i], 128);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(512u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===== TMA producer + tile scheduler =====
        // Tiles are claimed from a global counter: under HBM contention SMs progress at very different rates
        // (ncu: fastest SM done in 56 % of the time with a static split), so the split must be dynamic.
        if (lane == 0) {
            int stage = 0, it = 0;
            uint32_t phase = 0;
            for (;; ++it) {
                int tile = (int)atomicAdd(p.tile_counter, 1u);
                if (tile >= n_tiles) tile = -1;
                tile_q[it & (TC_TQ - 1)] = tile;                       // published by the next arrive on full[stage]
                if (tile < 0) {                              // end of work: an empty stage carries the sentinel
                    mbar_wait(&empty[stage], phase ^ 1);
                    mbar_arrive(&full[stage]);
                    break;
                }
                const int sub0 = tile * T;
                const int nv = min(T, n_sub - sub0);
                const uint64_t hint = 0x12F0000000000000ull;     // evict first: every sample is read once
                for (int c = 0; c < n_chunks; ++c) {
                    mbar_wait(&empty[stage], phase ^ 1);
                    unsigned char *dst = sA + stage * SM.a_stage;
                    if (use4d && (c + 1) * KC <= n_full) {
                        // one 4-D box {128 B, 8 frames, T spans, KC/8 groups}: the TMA walks the T adjacent spans of a
                        // frame back to back, so DRAM sees T*128 contiguous bytes per frame (the probe: 2 KB segments
                        // reach 7.0 TB/s where isolated 128-byte rows stop at 6.0)
                        mbar_expect_tx(&full[stage], (uint32_t)(SM.a_stage + SM.b_stage));
                        tma_load_4d(dst, &tmap4, &full[stage], 0, 0, sub0, c * (KC / GRP), hint);
                    } else {
                        // ragged tail in time (or a row pitch that is not a multiple of 128 B): 1 KB boxes, zero filled
                        // beyond the last frame / last byte
                        // groups wholly beyond the last frame are skipped: their digits are zero and integer 0 * stale = 0
                        const int ng = min(KC / GRP, (p.N - c * KC + GRP - 1) / GRP);
                        mbar_expect_tx(&full[stage], (uint32_t)(nv * ng * GRP * SUB_BYTES + SM.b_stage));
                        for (int g = 0; g < ng; ++g)
                            for (int t = 0; t < nv; ++t)
                                tma_load_2d(dst + (g * T + t) * (GRP * SUB_BYTES), &tmap2, &full[stage], (sub0 + t) * SUB_BYTES, c * KC + g * GRP, hint);
                    }
                    bulk_load(sB + stage * SM.b_stage, p.digits + (size_t)c * SM.b_stage, SM.b_stage, &full[stage]);
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer =====
        // instruction descriptor (cute::UMMA::InstrDescriptor): D = s32, A = u8 MN-major, B = s8 K-major, M = 128, N = NC
        constexpr uint32_t idesc = (2u << 4) | (0u << 7) | (1u << 10) | (1u << 15) | (0u << 16) | ((uint32_t)(NC >> 3) << 17) | ((128u >> 4) << 24);
        int stage = 0;
        uint32_t phase = 0;
        for (int it = 0;; ++it) {
            const int buf = it & 1;
            mbar_wait(&tempty[buf], ((it >> 1) & 1) ^ 1);     // epilogue has drained this accumulator buffer
            tc_fence_after();
            mbar_wait(&full[stage], phase);                   // first chunk of the tile (or the sentinel) has landed
            const int tile = tile_q[it & (TC_TQ - 1)];
            if (lane == 0) tbuf_tile[buf] = tile;
            if (tile < 0) {
                if (lane == 0) { mbar_arrive(&tfull[buf]); mbar_arrive(&tfull[buf]); }
                break;
            }
            const int nv = min(T, n_sub - tile * T);
            for (int c = 0; c < n_chunks; ++c) {
                if (c > 0) mbar_wait(&full[stage], phase);
                tc_fence_after();
                if (lane == 0) {
                    const uint32_t a0 = smem_u32(sA + stage * SM.a_stage), b0 = smem_u32(sB + stage * SM.b_stage);
                    for (int t = 0; t < nv; ++t) {
                        for (int ks = 0; ks < KC / MMA_K; ++ks) {
                            // A: MN-major, 128-byte swizzle: rows of 128 pixel bytes, 8-frame atoms T KB apart (SBO)
                            const uint64_t ad = smem_desc(a0 + (ks * (MMA_K / GRP) * T + t) * (GRP * SUB_BYTES), T * GRP * SUB_BYTES, T * GRP * SUB_BYTES, 2);
                            // B: K-major, no swizzle: K halves 128 B apart (LBO), 8-column groups 256 B apart (SBO)
                            const uint64_t bd = smem_desc(b0 + ks * NC * MMA_K, 128, 256, 0);
                            tc_mma_i8(tmem_base + (uint32_t)(buf * T * NC + t * NC), ad, bd, idesc, (c | ks) ? 1u : 0u);
                        }
                    }
                    tc_commit(&empty[stage]);                 // frees the stage when these MMAs have read it
                    if (c == n_chunks - 1) {
                        tc_commit(&tfull[buf]);               // arrival 1 of 2: the accumulators are complete
                        mbar_arrive(&tfull[buf]);             // arrival 2 of 2: releases tbuf_tile[buf]
                    }
                }
                __syncwarp();
                if (++stage == STAGES) { stage = 0; phase ^= 1; }
            }
        }
    } else {
        // ===== epilogue: TMEM -> registers -> exact int64 sums -> A4 finalise =====
        const int q = warp & 3;                         // TMEM lane quarter this warp may read
        const int m = q * 32 + lane;                    // accumulator row = byte index inside the 128-byte span
        for (int it = 0;; ++it) {
            const int buf = it & 1;
            mbar_wait(&tfull[buf], (it >> 1) & 1);
            const int tile = tbuf_tile[buf];
            if (tile < 0) break;
            const int nv = min(T, n_sub - tile * T);
            tc_fence_after();
            for (int t = 0; t < nv; ++t) {
                const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * T * NC + t * NC);
                const int64_t byte0 = (int64_t)(tile * T + t) * SUB_BYTES + m;
                const int64_t pixel = BYTES == 2 ? (byte0 >> 1) : byte0;
                const bool valid = byte0 < p.row_bytes;
#pragma unroll
                for (int g = 0; g < NC / 16; ++g) {       // 16 columns = 4 reference rows = 2 references per group
                    uint32_t r[16];
                    tc_ld16(taddr + g * 16, r);
                    tc_wait_ld();
                    long long v[4];
#pragma unroll
                    for (int rr = 0; rr < 4; ++rr)
                        v[rr] = (long long)(int)r[4 * rr] + ((long long)(int)r[4 * rr + 1] << 8) + ((long long)(int)r[4 * rr + 2] << 16) +
                                ((long long)(int)r[4 * rr + 3] << 24);
                    if (BYTES == 2) {
                        // even row = low byte, odd row = high byte of the same pixel: x = lo + 256 * hi
#pragma unroll
                        for (int rr = 0; rr < 4; ++rr) {
                            const long long o = __shfl_xor_sync(0xffffffffu, v[rr], 1);
                            v[rr] = (lane & 1) ? (o + (v[rr] << 8)) : (v[rr] + (o << 8));
                        }
                    }
                    // this group holds references 2g and 2g+1; with 16-bit samples the lane pair splits them
#pragma unroll
                    for (int kk = 0; kk < 2; ++kk) {
                        const int k = 2 * g + kk;
                        const bool mine = BYTES == 1 || (lane & 1) == kk;
                        if (valid && mine && k < p.fin.K) {
                            const long long Si = v[2 * kk], Ci = v[2 * kk + 1];
                            const int64_t o = (int64_t)k * p.HW + pixel;
                            if (p.sums_out) {
                                p.sums_out[(int64_t)(2 * k) * p.HW + pixel] = Si;
                                p.sums_out[(int64_t)(2 * k + 1) * p.HW + pixel] = Ci;
                            }
                            const double S = (double)Si * (p.fin.scale * 9.31322574615478515625e-10);   // 2^-30
                            const double C = (double)Ci * (p.fin.scale * 9.31322574615478515625e-10);
                            if (p.fin.I) p.fin.I[o] = (float)S;
                            if (p.fin.Q) p.fin.Q[o] = (float)C;
                            if (p.fin.amp) p.fin.amp[o] = (float)sqrt(S * S + C * C);
                            if (p.fin.phase) p.fin.phase[o] = (Si == 0 && Ci == 0) ? 0.0f : (float)atan2(C, S);
                        }
                    }
                }
            }
            tc_fence_before();
            mbar_arrive(&tempty[buf]);
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512u) : "memory");
    }
}

// Tile shape for (NC columns, frame size): T spans (T*128 contiguous bytes of every frame per CTA tile; the wider,
// the friendlier to DRAM), accumulators double buffered in the 512 TMEM columns; KC frames per stage; as many
// stages as fit in shared memory.
struct TcShape { int T, kc, stages, use4d; };

TcShape tc_shape(int nc, int64_t row_bytes, int N, int n_sms, const int *force)
{
    TcShape sh;
    const int n_sub = (int)((row_bytes + SUB_BYTES - 1) / SUB_BYTES);
    // Measured on cfg2 (B200): the tensor pipe takes about 200 cycles to fetch one MN-major 8-bit A tile (128 bytes x
    // 32 frames) from shared memory whatever N is, i.e. about 21 B/clk/SM = 6.1 TB/s over 148 SMs -- that, not HBM,
    // bounds this kernel.  64-frame stages (two MMAs per span per barrier round trip) and 1 KB of contiguous
    // bytes per frame were the best point of the sweep (T,stages,KC = 8,3,64: 6.17 TB/s; 16,3,32: 5.05; 4,6,64: 5.78).
    int T = 512 / (2 * nc);
    if (T > 8) T = 8;
    while (T & (T - 1)) --T;                                        // power of two
    while (T > 1 && (n_sub + T - 1) / T < 2 * n_sms) T /= 2;      // small frames: keep every SM busy
    sh.T = T;
    sh.kc = 64;
    sh.stages = (200 * 1024) / TcSmem(nc, T, 1, sh.kc).off_bar;
    if (force && force[0] > 0) {                          // debug / test override (qld_debug_set_tile): T, STAGES, KC
        const int t = force[0], s2 = force[1], kc = force[2];
        if (2 * t * nc <= 512 && s2 >= 2 && (kc == 32 || kc == 64) && TcSmem(nc, t, s2, kc).total + 1024 <= 227 * 1024) { sh.T = t; sh.stages = s2; sh.kc = kc; }
    }
    if (sh.stages > TC_MAX_STAGES) sh.stages = TC_MAX_STAGES;
    sh.use4d = (row_bytes % SUB_BYTES == 0 && N >= GRP) ? 1 : 0;
    return sh;
}

template <int NC, int BYTES>
cudaError_t launch_tc(const CUtensorMap *tmaps, const TcParams &p, int n_sms, cudaStream_t st)
{
    const int force[3] = {p.force_T, p.force_stages, p.force_kc};
    const TcShape sh = tc_shape(NC, p.row_bytes, p.N, n_sms, force);
    const TcSmem SM(NC, sh.T, sh.stages, sh.kc);
    auto kern = k_demod_tc<NC, BYTES>;
    // raise the kernel's dynamic shared-memory limit once per size (per instantiation; the attribute is per device
    // function, and re-setting it on every launch costs a driver call)
    static int smem_set_dev[64] = {0};
    int dev = 0;
    cudaGetDevice(&dev);
    int &smem_set = smem_set_dev[dev & 63];
    cudaError_t e = cudaSuccess;
    if (SM.total + 1024 > smem_set) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SM.total + 1024);
        if (e != cudaSuccess) return e;
        smem_set = SM.total + 1024;
    }
    const int n_sub = (int)((p.row_bytes + SUB_BYTES - 1) / SUB_BYTES);
    const int n_tiles = (n_sub + sh.T - 1) / sh.T;
    const int grid = n_tiles < n_sms ? n_tiles : n_sms;
    e = cudaMemsetAsync(p.tile_counter, 0, sizeof(unsigned int), st);
    if (e != cudaSuccess) return e;
    kern<<<grid, 192, SM.total + 1024, st>>>(tmaps[0], tmaps[1], p, sh.T, sh.stages, sh.kc, sh.use4d);
    return cudaGetLastError();
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace

int qld_tc_columns(int K) { const int c = 8 * K; return (c + 15) / 16 * 16; }

size_t qld_tc_digit_bytes(int K, int N)
{
    const int n_chunks = (N + KC_PAD - 1) / KC_PAD;
    return (size_t)n_chunks * (KC_PAD / MMA_K) * qld_tc_columns(K) * MMA_K;
}

// Two tensor maps over the frame stack, written to tmaps_out[0..1]:
//  [0] 2-D {row bytes, frames}, box {128 B, 8 frames}: one swizzle atom, any shape (zero fill beyond the edges);
//  [1] 4-D {128 B, 8 frames, spans, frame groups}, box {128, 8, T, KC/8}: a whole pipeline stage in one copy,
//      spans innermost in the walk.  Only valid (and only used) when row_bytes % 128 == 0 and N >= 8.
cudaError_t qld_tc_encode_tmap(void *tmaps_out, const void *frames, int64_t row_bytes, int n_frames, int K, int n_sms, const int *force)
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
    CUtensorMap *tm = reinterpret_cast<CUtensorMap *>(tmaps_out);
    {
        const cuuint64_t dims[2] = {(cuuint64_t)row_bytes, (cuuint64_t)n_frames};
        const cuuint64_t strides[1] = {(cuuint64_t)row_bytes};
        const cuuint32_t box[2] = {SUB_BYTES, GRP};
        const cuuint32_t estr[2] = {1, 1};
        CUresult r = fn(&tm[0], CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void *>(frames), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
    }
    const TcShape sh = tc_shape(qld_tc_columns(K), row_bytes, n_frames, n_sms, force);
    if (sh.use4d) {
        const cuuint64_t dims[4] = {SUB_BYTES, GRP, (cuuint64_t)(row_bytes / SUB_BYTES), (cuuint64_t)(n_frames / GRP)};
        const cuuint64_t strides[3] = {(cuuint64_t)row_bytes, SUB_BYTES, (cuuint64_t)row_bytes * GRP};
        const cuuint32_t box[4] = {SUB_BYTES, GRP, (cuuint32_t)sh.T, (cuuint32_t)(sh.kc / GRP)};
        const cuuint32_t estr[4] = {1, 1, 1, 1};
        CUresult r = fn(&tm[1], CU_TENSOR_MAP_DATA_TYPE_UINT8, 4, const_cast<void *>(frames), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
    } else {
        tm[1] = tm[0];
    }
    return cudaSuccess;
}

cudaError_t qld_launch_fixed_table_fill(const TableFillParams &p, int32_t *rfix, int n_stride, cudaStream_t st)
{
    k_fixed_table_fill<<<(p.n * p.K + 255) / 256, 256, 0, st>>>(p, rfix, n_stride);
    return cudaGetLastError();
}

cudaError_t qld_launch_fixed_from_doubles(const double *tab, int n, int k, int32_t *rfix, int n_stride, cudaStream_t st)
{
    k_fixed_from_doubles<<<(n + 255) / 256, 256, 0, st>>>(tab, n, k, rfix, n_stride);
    return cudaGetLastError();
}

cudaError_t qld_launch_digit_pack(const int32_t *rfix, int n_stride, int N, int K, int8_t *digits, cudaStream_t st)
{
    const int nc = qld_tc_columns(K);
    const int n_steps = (N + KC_PAD - 1) / KC_PAD * (KC_PAD / MMA_K);
    const int64_t total = (int64_t)n_steps * nc * MMA_K;
    k_digit_pack<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(rfix, n_stride, N, 2 * K, nc, n_steps, digits);
    return cudaGetLastError();
}

cudaError_t qld_launch_demod_tc(const void *tmaps, const TcParams &p, int n_sms, cudaStream_t st)
{
    const CUtensorMap *tm = reinterpret_cast<const CUtensorMap *>(tmaps);
    const int nc = qld_tc_columns(p.fin.K);
    if (p.bytes == 2) {
        switch (nc) {
        case 16: return launch_tc<16, 2>(tm, p, n_sms, st);
        case 32: return launch_tc<32, 2>(tm, p, n_sms, st);
        case 48: return launch_tc<48, 2>(tm, p, n_sms, st);
        case 64: return launch_tc<64, 2>(tm, p, n_sms, st);
        }
    } else {
        switch (nc) {
        case 16: return launch_tc<16, 1>(tm, p, n_sms, st);
        case 32: return launch_tc<32, 1>(tm, p, n_sms, st);
        case 48: return launch_tc<48, 1>(tm, p, n_sms, st);
        case 64: return launch_tc<64, 1>(tm, p, n_sms, st);
        }
    }
    return cudaErrorInvalidValue;
}

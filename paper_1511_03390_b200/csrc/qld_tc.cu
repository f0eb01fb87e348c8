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
// The kernel is HBM-bound for any K <= 8 (N columns = 8K <= 64): measured, an M = 128, N <= 128, K = 32 kind::i8 MMA retires in
// about 40 ns (MN-major and K-major operands alike), i.e. 4 KB of samples per 40 ns per SM, twice what HBM delivers to one SM --
// PROVIDED the MMA warp issues warp-uniformly (see the MMA issuer below).
//
// The same kernel runs two more contractions (template MODE): the integer phase bins of A3' (MODE 1: the bin indicators 0, +-1
// are a one-digit B operand of 16 columns, the epilogue writes the exact int32 rows) and the unknown-frequency search (MODE 2:
// 32 DFT bins = 256 columns per launch, arg-max in the epilogue; qld_spectrum.cu).
//
// Structure (one persistent CTA per SM, 320 threads): warp 0 = TMA producer, warp 1 = MMA issuer, warps 2-9 =
// epilogue (TMEM -> registers -> maps; two quartets, each warp reads its own TMEM lane quarter).  A CTA tile is T adjacent
// 128-byte pixel spans over all frames.  When two
// tiles' accumulators fit the 512 TMEM columns (2 * T * NC <= 512) they are double buffered; otherwise (K = 8: NC = 64,
// T = 8 -- 1 KB of contiguous bytes per frame, which DRAM serves measurably better than 512 B) there is one set and the
// epilogue hands the columns back span by span: the MMA warp restarts span t of the next tile as soon as span t is
// drained, and the TMA producer keeps filling the stage ring meanwhile, so HBM never idles.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "qld_angle.cuh"
#include "qld_internal.h"
#include "qld_ptx.cuh"
#include "qld_tc.h"

using namespace qld_ptx;
using qld_angle::half_turns_of;

// tile shape of the unknown-frequency search (256 columns): T = 2 spans share every digit tile (the digit tiles are twice the
// bytes of a span's frames: with T = 1 the L2 -> shared-memory traffic, three times the HBM traffic, is the bound), one
// accumulator set handed back span by span
#define QLD_SPEC_T 2
#define QLD_SPEC_STAGES 3

namespace {

constexpr int KC_PAD = 64;        // the digit tiles are padded to a multiple of this many frames
constexpr int SUB_BYTES = 128;    // pixel bytes per MMA M tile
constexpr int MMA_K = 32;         // frames per tcgen05.mma (8-bit operands)
constexpr int GRP = 8;            // frames per 128-byte-swizzle atom (8 rows of 128 bytes = 1 KB)
constexpr int TC_TQ = 16;         // tile-id queue entries: the producer runs at most `stages` <= 12 tiles ahead of the MMA warp
constexpr int TC_MAX_STAGES = 12;
constexpr int EPI_SETS = 2;        // epilogue warp quartets: set e drains the spans t with t % EPI_SETS == e
constexpr int TC_THREADS = 64 + 128 * EPI_SETS;
constexpr int TC_MAX_SPANS = 32;  // accumulator sets: T spans, times two when double buffered
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
// one lane of the (fully active) warp; the compiler keeps values that do not depend on the lane in uniform registers, which
// is what tcgen05.mma's descriptor operands want
__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.b32 %0, 1, 0, P;\n\t}" : "=r"(pred));
    return pred != 0;
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

// B operand of the integer-bin contraction: the same [step][n/8][k/16][n%8][k%16] tiles with 16 columns, column c = bin row c,
// one signed byte (0, +1, -1) per frame
__global__ void k_bins_pack(const int32_t *wtab, int cap_w, int rows, int n, int n_steps, int8_t *digits)
{
    constexpr int nc = 16;
    const int64_t total = (int64_t)n_steps * nc * MMA_K;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int q = (int)(idx / (nc * MMA_K));
        const int rem = (int)(idx % (nc * MMA_K));
        const int k0 = rem & 15, n0 = (rem >> 4) & 7, k1 = (rem >> 7) & 1, n1 = rem >> 8;
        const int c = n1 * 8 + n0, s = q * MMA_K + k1 * 16 + k0;          // frame s + 1
        int d = 0;
        if (s < n && c < rows) d = wtab[(int64_t)((s + 1) % cap_w) * rows + c];
        digits[idx] = (int8_t)d;
    }
}

// Digit tiles of the unknown-frequency search: pass P holds the DFT bins q_lo + 32 P .. (nu = q / N, reduced exactly as
// (q s) mod N), 256 columns: column c = 4 * (2 * b + row) + j = digit j of sin (row 0) / cos (row 1) of bin b of the pass.
// Steps (32 frames) are padded to a multiple of 4: the search runs 128-frame stages.
__global__ void k_spectrum_digits(int N, int q_lo, int n_bins, int n_steps, int8_t *digits)
{
    constexpr int nc = 256;
    const int n_pass = (n_bins + 31) / 32;
    const int64_t total = (int64_t)n_pass * n_steps * nc * MMA_K;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int P = (int)(idx / ((int64_t)n_steps * nc * MMA_K));
        const int64_t in_pass = idx % ((int64_t)n_steps * nc * MMA_K);
        const int q = (int)(in_pass / (nc * MMA_K));
        const int rem = (int)(in_pass % (nc * MMA_K));
        const int k0 = rem & 15, n0 = (rem >> 4) & 7, k1 = (rem >> 7) & 1, n1 = rem >> 8;
        const int c = n1 * 8 + n0, s = q * MMA_K + k1 * 16 + k0;          // frame s + 1
        const int b = c >> 3, row = (c >> 2) & 1, j = c & 3;
        const int bin = P * 32 + b;
        int d = 0;
        if (s < N && bin < n_bins) {
            const uint64_t r = ((uint64_t)(q_lo + bin) * (uint64_t)(s + 1)) % (uint64_t)N;
            double sn, cs;
            sincospi(2.0 * (double)r / (double)N, &sn, &cs);
            int32_t v = (int32_t)rint((row ? cs : sn) * 1073741824.0);
            for (int t = 0; t <= j; ++t) {
                d = ((v + 128) & 255) - 128;
                v = (v - d) >> 8;
            }
        }
        digits[idx] = (int8_t)d;
    }
}

// ---------------------------------------------------------------------------------------------------
// the contraction kernel
// ---------------------------------------------------------------------------------------------------
// sqrt of a non-negative double to a few units in 1e-14: fp32 reciprocal square root of the rounded argument, one Newton
// step in fp64 (the library routine is correctly rounded but several times longer; the result is stored as fp32)
__device__ __forceinline__ double sqrt_newton(double x)
{
    if (x == 0.0) return 0.0;
    const double y = (double)rsqrtf((float)x);
    const double r = x * y;
    return fma(0.5 * y, fma(-r, r, x), r);
}

// A4 for one pixel of one reference from its exact sums (I * 2^30, Q * 2^30)
__device__ __forceinline__ void emit_fixed(const TcParams &p, int k, int64_t pixel, long long Si, long long Ci, double sc30)
{
    const int64_t o = (int64_t)k * p.HW + pixel;
    if (p.sums_out) {
        p.sums_out[(int64_t)(2 * k) * p.HW + pixel] = Si;
        p.sums_out[(int64_t)(2 * k + 1) * p.HW + pixel] = Ci;
    }
    const double S = (double)Si * sc30, C = (double)Ci * sc30;
    if (p.fin.I) p.fin.I[o] = (float)S;
    if (p.fin.Q) p.fin.Q[o] = (float)C;
    if (p.fin.amp) p.fin.amp[o] = (float)sqrt_newton(fma(S, S, C * C));
    if (p.fin.phase) p.fin.phase[o] = (Si == 0 && Ci == 0) ? 0.0f : (float)atan2(C, S);
}

// shared-memory carve-up for (NC columns, T spans per tile, STAGES pipeline stages)
struct TcSmem {
    int a_stage, b_stage, off_b, off_bar, total;
    __host__ __device__ TcSmem(int nc, int t, int stages, int kc)
    {
        a_stage = t * kc * SUB_BYTES;                 // [kc/8 frame groups][t spans][8 frames][128 bytes]
        b_stage = (kc / MMA_K) * nc * MMA_K;
        off_b = stages * a_stage;
        off_bar = off_b + stages * b_stage;
        total = off_bar + (2 * stages + 2 + TC_MAX_SPANS) * 8 + 16 + 8 + TC_TQ * 4 + 8 + 2 * 192 * 8;   // barriers, TMEM slot, tile queue, tbuf_tile, search exchange
    }
};

// TT, KCC > 0: the tile shape as compile-time constants (the shape the launcher picks for large frames): the MMA warp's
// loops over spans and K steps unroll and every descriptor is "stage base + immediate"; 0: run-time shape (T_rt, KC_rt).
// MODE: 0 = fixed-point references (A3 / A6), 1 = integer phase bins (A3'), 2 = unknown-frequency search (32 DFT bins per launch)
template <int NC, int BYTES, int TT, int KCC, int MODE>
__global__ void __launch_bounds__(TC_THREADS, 1) k_demod_tc(const __grid_constant__ CUtensorMap tmap2, const __grid_constant__ CUtensorMap tmap4,
                                                     const TcParams p, const int T_rt, const int STAGES, const int KC_rt, const int use4d)
{
    const int T = TT > 0 ? TT : T_rt, KC = KCC > 0 ? KCC : KC_rt;
    const TcSmem SM(NC, T, STAGES, KC);
    extern __shared__ unsigned char smem_raw[];
    // 128-byte-swizzled TMA/UMMA tiles need 1024-byte alignment in the shared window
    unsigned char *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    unsigned char *sA = smem;
    unsigned char *sB = smem + SM.off_b;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + SM.off_bar);
    uint64_t *empty = full + STAGES;
    uint64_t *tfull = empty + STAGES;
    uint64_t *tempty = tfull + 2;                       // [NBUF * T] one per span accumulator: drained by the epilogue
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tempty + TC_MAX_SPANS);
    volatile int *tile_q = reinterpret_cast<volatile int *>(tmem_slot + 2);      // [TC_TQ] tile ids, producer -> MMA warp
    volatile int *tbuf_tile = tile_q + TC_TQ;                                        // [2] tile id per accumulator buffer
    double *spec_x = reinterpret_cast<double *>(const_cast<int *>(tbuf_tile) + 2);     // [2][192] search mode: quartet 1 -> quartet 0

    // the warp index as a broadcast: the compiler then knows that the role branches below are warp-uniform and keeps the MMA
    // warp's loop state in uniform registers
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
    const int n_chunks = (p.N + KC - 1) / KC;
    const int n_full = p.N / GRP * GRP;               // frames covered by whole 8-frame groups (the 4-D map's extent)
    const int n_sub = (int)((p.row_bytes + SUB_BYTES - 1) / SUB_BYTES);
    const int n_tiles = (n_sub + T - 1) / T;
    const int NBUF = 2 * T * NC <= 512 ? 2 : 1;       // accumulator sets in TMEM

    if (threadIdx.x == 0) {
        if (blockIdx.x == 0) *p.tile_counter_next = 0;
        for (int i = 0; i < STAGES; ++i) {
            mbar_init(&full[i], 1);
            mbar_init(&empty[i], 1);
        }
        for (int i = 0; i < 2; ++i) mbar_init(&tfull[i], 2);
        for (int i = 0; i < TC_MAX_SPANS; ++i) mbar_init(&tempty[i], MODE == 2 ? 128 * EPI_SETS : 128);   // search mode: both quartets drain every span
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(512u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot, 0);      // broadcast: provably warp-uniform

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
        // The whole warp runs this loop and one elected lane issues: every operand of tcgen05.mma (descriptors, TMEM address)
        // is then warp-uniform and lives in uniform registers.  Under `if (lane == 0)` the compiler cannot prove that and
        // wraps every MMA in an ELECT / 5 x R2UR / branch sequence of about 200 cycles -- which, not the operand fetch, was
        // what held the round-1 kernel at 20 bytes per clock per SM (an MMA of this shape retires in about 80 cycles).
        // instruction descriptor (cute::UMMA::InstrDescriptor): D = s32, A = u8 MN-major, B = s8 K-major, M = 128, N = NC
        constexpr uint32_t idesc = (2u << 4) | (0u << 7) | (1u << 10) | (1u << 15) | (0u << 16) | ((uint32_t)(NC >> 3) << 17) | ((128u >> 4) << 24);
        const bool leader = elect_one();
        const uint32_t sA0 = smem_u32(sA), sB0 = smem_u32(sB);
        const uint32_t a_sbo = (uint32_t)(T * GRP * SUB_BYTES);
        int stage = 0;
        uint32_t phase = 0;
        for (int it = 0;; ++it) {
            const int buf = it & 1;                           // hand-off slot (tfull / tbuf_tile), always alternating
            const int abuf = NBUF == 2 ? buf : 0;             // accumulator set
            const uint32_t epar = (NBUF == 2 ? (uint32_t)(it >> 1) : (uint32_t)it) & 1u;   // a set's barriers flip once per use
            mbar_wait(&full[stage], phase);                   // first chunk of the tile (or the sentinel) has landed
            const int tile = __shfl_sync(0xffffffffu, tile_q[it & (TC_TQ - 1)], 0);
            // The first span of every epilogue quartet (spans 0 .. EPI_SETS-1 of this accumulator set) is drained: each
            // quartet is then past the hand-off that used tfull[buf] / tbuf_tile[buf] two tiles ago, so both may be reused.
            for (int e = 0; e < (MODE == 2 ? 1 : EPI_SETS) && e < T; ++e) mbar_wait(&tempty[abuf * T + e], epar ^ 1u);
            if (leader) tbuf_tile[buf] = tile;
            if (tile < 0) {
                if (leader) { mbar_arrive(&tfull[buf]); mbar_arrive(&tfull[buf]); }
                break;
            }
            const int nv = min(T, n_sub - tile * T);
            const uint32_t d0 = tmem_base + (uint32_t)(abuf * T * NC);
            for (int c = 0; c < n_chunks; ++c) {
                if (c > 0) mbar_wait(&full[stage], phase);
                tc_fence_after();
                // descriptors of this stage: A MN-major with 128-byte swizzle (rows of 128 pixel bytes, 8-frame atoms T KB
                // apart = SBO); B K-major without swizzle (K halves 128 B apart = LBO, 8-column groups 256 B apart = SBO).
                // The start address sits in the low 14 bits (units of 16 bytes): span t / K step ks are plain additions.
                const uint64_t ad0 = smem_desc(sA0 + (uint32_t)(stage * SM.a_stage), a_sbo, a_sbo, 2);
                const uint64_t bd0 = smem_desc(sB0 + (uint32_t)(stage * SM.b_stage), 128, 256, 0);
                if (TT > 0) {
#pragma unroll
                    for (int t = 0; t < (TT > 0 ? TT : 1); ++t) {
                        if (t < nv) {
                            if (c == 0) {                     // the epilogue has drained this span's previous accumulator
                                mbar_wait(&tempty[abuf * T + t], epar ^ 1u);
                                tc_fence_after();
                            }
#pragma unroll
                            for (int ks = 0; ks < (KCC > 0 ? KCC : MMA_K) / MMA_K; ++ks) {
                                const uint64_t ad = ad0 + (uint64_t)(((ks * (MMA_K / GRP) * TT + t) * (GRP * SUB_BYTES)) >> 4);
                                const uint64_t bd = bd0 + (uint64_t)((ks * NC * MMA_K) >> 4);
                                if (leader) tc_mma_i8(d0 + (uint32_t)(t * NC), ad, bd, idesc, (c | ks) ? 1u : 0u);
                            }
                        }
                    }
                } else {
                    for (int t = 0; t < nv; ++t) {
                        if (c == 0) {
                            mbar_wait(&tempty[abuf * T + t], epar ^ 1u);
                            tc_fence_after();
                        }
                        for (int ks = 0; ks < KC / MMA_K; ++ks) {
                            const uint64_t ad = ad0 + (uint64_t)(((ks * (MMA_K / GRP) * T + t) * (GRP * SUB_BYTES)) >> 4);
                            const uint64_t bd = bd0 + (uint64_t)((ks * NC * MMA_K) >> 4);
                            if (leader) tc_mma_i8(d0 + (uint32_t)(t * NC), ad, bd, idesc, (c | ks) ? 1u : 0u);
                        }
                    }
                }
                if (leader) {
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
        const int eset = (warp - 2) >> 2;               // which quartet of epilogue warps: it drains spans t % EPI_SETS == eset
        const int m = q * 32 + lane;                    // accumulator row = byte index inside the 128-byte span
        int span_seq = 0;                               // search mode: spans this CTA has reduced so far (both quartets count alike)
        for (int it = 0; MODE == 2 || eset < T; ++it) { // a quartet without spans (T < EPI_SETS) has nothing to do
            const int buf = it & 1;
            const int abuf = NBUF == 2 ? buf : 0;
            mbar_wait(&tfull[buf], (it >> 1) & 1);
            const int tile = tbuf_tile[buf];
            if (tile < 0) break;
            const int nv = min(T, n_sub - tile * T);
            tc_fence_after();
            for (int t = (MODE == 2 ? 0 : eset); t < T; t += (MODE == 2 ? 1 : EPI_SETS)) {
                if (t >= nv) {                                // span beyond the frame: nothing was accumulated, hand it back
                    mbar_arrive(&tempty[abuf * T + t]);
                    continue;
                }
                const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(abuf * T * NC + t * NC);
                const int64_t byte0 = (int64_t)(tile * T + t) * SUB_BYTES + m;
                const int64_t pixel = BYTES == 2 ? (byte0 >> 1) : byte0;
                const bool valid = byte0 < p.row_bytes;
                if constexpr (MODE == 2) {
                    // unknown-frequency search: 32 bins = 16 groups of 16 columns; quartet e takes the groups g = e mod 2.  The
                    // squared amplitude of every bin is compared in fp64 against the thread's running best (strictly greater:
                    // the lowest bin wins a tie); the two quartets meet through shared memory, then one read-modify-write of
                    // the maps that persist across the passes.
                    double best = -1.0;
                    int best_q = 0;
                    // the running maximum of earlier passes is requested now and used at the very end
                    const bool writer = eset == 0 && valid && (BYTES == 1 || !(lane & 1));
                    float prev_amp = -1.0f;
                    if (writer && !p.spec_first) prev_amp = __ldg(p.spec_amp + pixel);
                    uint32_t rn[16];
                    tc_ld16(taddr + eset * 16, rn);                             // software pipeline: the next group's columns are in flight
                    for (int g = eset; g < NC / 16; g += EPI_SETS) {
                        uint32_t r[16];
                        tc_wait_ld();
#pragma unroll
                        for (int i = 0; i < 16; ++i) r[i] = rn[i];
                        if (g + EPI_SETS < NC / 16) tc_ld16(taddr + (g + EPI_SETS) * 16, rn);
                        long long v[4];
#pragma unroll
                        for (int rr = 0; rr < 4; ++rr)
                            v[rr] = (long long)(int)r[4 * rr] + ((long long)(int)r[4 * rr + 1] << 8) + ((long long)(int)r[4 * rr + 2] << 16) +
                                    ((long long)(int)r[4 * rr + 3] << 24);
                        if (BYTES == 2) {
#pragma unroll
                            for (int rr = 0; rr < 4; ++rr) {
                                const long long o = __shfl_xor_sync(0xffffffffu, v[rr], 1);
                                v[rr] = (((lane & 1) != 0) != (p.big_endian != 0)) ? (o + (v[rr] << 8)) : (v[rr] + (o << 8));
                            }
                        }
#pragma unroll
                        for (int kk = 0; kk < 2; ++kk) {
                            if (BYTES == 2 && (lane & 1) != kk) continue;      // the lane pair of a 16-bit pixel splits the two bins
                            const int b = 2 * g + kk;
                            const double S = (double)v[2 * kk], C = (double)v[2 * kk + 1];
                            const double a2 = fma(S, S, C * C);
                            if (b < p.spec_nbins && a2 > best) { best = a2; best_q = p.spec_q0 + b; }
                        }
                    }
                    tc_fence_before();
                    mbar_arrive(&tempty[abuf * T + t]);
                    if (BYTES == 2) {                                           // even bins sit in the even lane, odd bins in the odd lane
                        const double ob = __shfl_xor_sync(0xffffffffu, best, 1);
                        const int oq = __shfl_xor_sync(0xffffffffu, best_q, 1);
                        if (ob > best || (ob == best && oq < best_q)) { best = ob; best_q = oq; }
                    }
                    // 128 doubles + 128 ints per buffer; the buffers alternate from span to span (not from tile to tile: with one
                    // barrier per span, quartet 1 would otherwise write span t + 1 into the buffer quartet 0 still reads for span t)
                    double *sx = spec_x + (size_t)(span_seq++ & 1) * 192;
                    if (eset == 1) { sx[m] = best; reinterpret_cast<int *>(sx + 128)[m] = best_q; }
                    named_barrier(2, 128 * EPI_SETS);
                    if (eset == 0) {
                        const double ob = sx[m];
                        const int oq = reinterpret_cast<const int *>(sx + 128)[m];
                        if (ob > best || (ob == best && oq < best_q)) { best = ob; best_q = oq; }
                        if (writer && best >= 0.0) {
                            const float amp = (float)(sqrt_newton(best) * (p.fin.scale * 9.31322574615478515625e-10));
                            if (p.spec_first || amp > prev_amp) { p.spec_amp[pixel] = amp; p.spec_bin[pixel] = best_q; }
                        }
                    }
                    continue;
                }
                // all NC columns of the span into registers with one wait, then the span goes straight back to the MMA warp:
                // the arithmetic below runs out of registers while the next tile's MMAs already overwrite the columns
                uint32_t r[NC / 16][16];
#pragma unroll
                for (int g = 0; g < NC / 16; ++g) tc_ld16(taddr + g * 16, r[g]);
                tc_wait_ld();
                tc_fence_before();
                mbar_arrive(&tempty[abuf * T + t]);
                if constexpr (MODE == 1) {
                    // integer phase bins (A3'): column c = bin row c, exact int32; the lane pair of a 16-bit pixel holds its
                    // low-byte and high-byte sums: bin = lo + 256 * hi
                    int bins[16];
#pragma unroll
                    for (int c = 0; c < 16; ++c) {
                        int v = (int)r[0][c];
                        if (BYTES == 2) {
                            const int o = __shfl_xor_sync(0xffffffffu, v, 1);
                            v = (((lane & 1) != 0) != (p.big_endian != 0)) ? (o + (v << 8)) : (v + (o << 8));
                        }
                        bins[c] = v;
                    }
                    if (valid) {
                        const FinParams &f = p.fin;
                        const bool odd = BYTES == 2 && (lane & 1);         // the lane pair shares the stores
#pragma unroll
                        for (int c = 0; c < 16; ++c)
                            if (c < p.bins_rows && (BYTES == 1 || ((c & 1) != 0) == odd)) p.bins_out[(int64_t)c * p.bins_stride + pixel] = bins[c];
                        for (int k = 0; k < f.K; ++k) {
                            const int off = f.row_off[k], end = off + f.n_rows[k];
                            double S = 0.0, C = 0.0;
#pragma unroll
                            for (int c = 0; c < 16; ++c)
                                if (c >= off && c < end) {
                                    S = fma((double)bins[c], f.sw[c], S);
                                    C = fma((double)bins[c], f.cw[c], C);
                                }
                            if (f.rot) {
                                const double rc = f.rot[2 * k], rs = f.rot[2 * k + 1], S2 = S * rc - C * rs;
                                C = C * rc + S * rs;
                                S = S2;
                            }
                            S *= f.scale;
                            C *= f.scale;
                            const int64_t o = (int64_t)k * p.HW + pixel;
                            if (BYTES == 1 || !odd) {
                                if (f.I) f.I[o] = (float)S;
                                if (f.amp) f.amp[o] = (float)sqrt(S * S + C * C);
                            }
                            if (BYTES == 1 || odd) {
                                if (f.Q) f.Q[o] = (float)C;
                                if (f.phase) f.phase[o] = (S == 0.0 && C == 0.0) ? 0.0f : (float)atan2(C, S);
                            }
                        }
                    }
                    continue;
                }
                const double sc30 = p.fin.scale * 9.31322574615478515625e-10;                   // scale * 2^-30
#pragma unroll
                for (int g = 0; g < NC / 16; ++g) {       // 16 columns = 4 reference rows = 2 references per group
                    long long v[4];
#pragma unroll
                    for (int rr = 0; rr < 4; ++rr)
                        v[rr] = (long long)(int)r[g][4 * rr] + ((long long)(int)r[g][4 * rr + 1] << 8) + ((long long)(int)r[g][4 * rr + 2] << 16) +
                                ((long long)(int)r[g][4 * rr + 3] << 24);
                    if (BYTES == 2) {
                        // even row = low byte, odd row = high byte of the same pixel (the other way round for QLD_U16_BE): x = lo + 256 * hi
#pragma unroll
                        for (int rr = 0; rr < 4; ++rr) {
                            const long long o = __shfl_xor_sync(0xffffffffu, v[rr], 1);
                            v[rr] = (((lane & 1) != 0) != (p.big_endian != 0)) ? (o + (v[rr] << 8)) : (v[rr] + (o << 8));
                        }
                    }
                    // this group holds references 2g and 2g+1; with 16-bit samples the lane pair splits them
                    if (BYTES == 2) {
                        const int k = 2 * g + (lane & 1);
                        const long long Si = (lane & 1) ? v[2] : v[0], Ci = (lane & 1) ? v[3] : v[1];
                        if (valid && k < p.fin.K) emit_fixed(p, k, pixel, Si, Ci, sc30);
                    } else {
#pragma unroll
                        for (int kk = 0; kk < 2; ++kk)
                            if (valid && 2 * g + kk < p.fin.K) emit_fixed(p, 2 * g + kk, pixel, v[2 * kk], v[2 * kk + 1], sc30);
                    }
                }
            }
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
    // T spans (T * 128 contiguous bytes of every frame) per tile and 64-frame stages: on large frames 1 KB per frame (T = 8) is
    // what DRAM serves best (6.2 TB/s against 5.6 for 512 B; the kernel is HBM-bound once the MMA warp issues warp-uniformly).
    // On frames with only a few tiles per SM the last round of equal tiles leaves SMs idle, so T is the power of two that
    // minimises rounds * (T + 1) -- the "+ 1" standing for the per-tile cost of ramp and epilogue -- larger T winning ties.
    int Tmax = 512 / nc;                                            // one accumulator set may fill the TMEM (K = 8: T = 8)
    if (Tmax > 8) Tmax = 8;
    while (Tmax & (Tmax - 1)) --Tmax;                               // power of two
    int T = Tmax;
    long best = -1;
    for (int t = Tmax; t >= 1; t /= 2) {
        const long tiles = (n_sub + t - 1) / t, rounds = (tiles + n_sms - 1) / n_sms;
        const long cost = rounds * (t + 1);
        if (best < 0 || cost < best) { best = cost; T = t; }
    }
    sh.T = T;
    sh.kc = 64;
    sh.stages = (225 * 1024) / TcSmem(nc, T, 1, sh.kc).off_bar;
    if (force && force[0] > 0) {                          // debug / test override (qld_debug_set_tile): T, STAGES, KC
        const int t = force[0], s2 = force[1], kc = force[2];
        if (t * nc <= 512 && t <= TC_MAX_SPANS / 2 && s2 >= 2 && (kc == 32 || kc == 64 || kc == 128) && TcSmem(nc, t, s2, kc).total + 1024 <= 227 * 1024) { sh.T = t; sh.stages = s2; sh.kc = kc; }
    }
    if (sh.stages > TC_MAX_STAGES) sh.stages = TC_MAX_STAGES;
    sh.use4d = (row_bytes % SUB_BYTES == 0 && N >= GRP) ? 1 : 0;
    return sh;
}

template <int NC, int BYTES, int TT, int KCC, int MODE>
cudaError_t launch_tc_shape(const CUtensorMap *tmaps, const TcParams &p, const TcShape &sh, int n_sms, cudaStream_t st)
{
    const TcSmem SM(NC, sh.T, sh.stages, sh.kc);
    auto kern = k_demod_tc<NC, BYTES, TT, KCC, MODE>;
    static std::atomic<int> smem_ok[64];                  // per instantiation (qld_allow_max_smem)
    cudaError_t e = qld_allow_max_smem(kern, smem_ok);
    if (e != cudaSuccess) return e;
    const int n_sub = (int)((p.row_bytes + SUB_BYTES - 1) / SUB_BYTES);
    const int n_tiles = (n_sub + sh.T - 1) / sh.T;
    const int grid = n_tiles < n_sms ? n_tiles : n_sms;
    kern<<<grid, TC_THREADS, SM.total + 1024, st>>>(tmaps[0], tmaps[1], p, sh.T, sh.stages, sh.kc, sh.use4d);
    return cudaGetLastError();
}

template <int NC, int BYTES, int MODE = 0>
cudaError_t launch_tc(const CUtensorMap *tmaps, const TcParams &p, int n_sms, cudaStream_t st)
{
    const int force[3] = {p.force_T, p.force_stages, p.force_kc};
    const TcShape sh = tc_shape(NC, p.row_bytes, p.N, n_sms, force);
    // the shape of large frames (T = 8 spans = 1 KB of every frame, 64-frame stages) has its own instantiation
    if (sh.T == 8 && sh.kc == 64) return launch_tc_shape<NC, BYTES, 8, 64, MODE>(tmaps, p, sh, n_sms, st);
    if constexpr (MODE == 1) {                              // integer bins on mid-size frames (BASELINE.json configs[1]): T = 4 unrolled too
        if (sh.T == 4 && sh.kc == 64) return launch_tc_shape<NC, BYTES, 4, 64, MODE>(tmaps, p, sh, n_sms, st);
    }
    return launch_tc_shape<NC, BYTES, 0, 0, MODE>(tmaps, p, sh, n_sms, st);
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

size_t qld_tc_spectrum_digit_bytes(int N, int n_bins, size_t *pass_bytes)
{
    const int n_steps = ((N + 127) / 128) * 4;
    const size_t per_pass = (size_t)n_steps * 256 * MMA_K;
    if (pass_bytes) *pass_bytes = per_pass;
    return per_pass * (size_t)((n_bins + 31) / 32);
}

cudaError_t qld_launch_spectrum_digits(int N, int q_lo, int n_bins, int8_t *digits, cudaStream_t st)
{
    const int n_steps = ((N + 127) / 128) * 4;
    const int64_t total = (int64_t)((n_bins + 31) / 32) * n_steps * 256 * MMA_K;
    k_spectrum_digits<<<(unsigned)((total + 255) / 256 < 65535 * 16 ? (total + 255) / 256 : 65535 * 16), 256, 0, st>>>(N, q_lo, n_bins, n_steps, digits);
    return cudaGetLastError();
}

// one pass of the search: 32 bins, 256 columns, QLD_SPEC_T spans per tile, 128-frame stages (the shape the tensor maps must have
// been encoded for: qld_tc_spectrum_shape)
void qld_tc_spectrum_shape(int force_out[3]) { force_out[0] = QLD_SPEC_T; force_out[1] = QLD_SPEC_STAGES; force_out[2] = 128; }

cudaError_t qld_launch_demod_tc_spectrum(const void *tmaps, const TcParams &p, int n_sms, cudaStream_t st)
{
    const CUtensorMap *tm = reinterpret_cast<const CUtensorMap *>(tmaps);
    const int force[3] = {QLD_SPEC_T, QLD_SPEC_STAGES, 128};
    const TcShape sh = tc_shape(256, p.row_bytes, p.N, n_sms, force);
    if (sh.T != QLD_SPEC_T || sh.kc != 128) return cudaErrorInvalidValue;
    return p.bytes == 2 ? launch_tc_shape<256, 2, QLD_SPEC_T, 128, 2>(tm, p, sh, n_sms, st) : launch_tc_shape<256, 1, QLD_SPEC_T, 128, 2>(tm, p, sh, n_sms, st);
}

cudaError_t qld_launch_bins_pack(const int32_t *wtab, int cap_w, int rows, int N, int8_t *digits, cudaStream_t st)
{
    const int n_steps = (N + KC_PAD - 1) / KC_PAD * (KC_PAD / MMA_K);
    const int64_t total = (int64_t)n_steps * 16 * MMA_K;
    k_bins_pack<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(wtab, cap_w, rows, N, n_steps, digits);
    return cudaGetLastError();
}

cudaError_t qld_launch_demod_tc(const void *tmaps, const TcParams &p, int n_sms, cudaStream_t st)
{
    const CUtensorMap *tm = reinterpret_cast<const CUtensorMap *>(tmaps);
    if (p.bins_rows > 0) return p.bytes == 2 ? launch_tc<16, 2, 1>(tm, p, n_sms, st) : launch_tc<16, 1, 1>(tm, p, n_sms, st);
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

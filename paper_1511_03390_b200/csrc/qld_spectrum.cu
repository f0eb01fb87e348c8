// Unknown-frequency search: the paper's Fourier decomposition "is essentially a series of QLDs being
// performed at different frequencies", and the FFT image is |F(j,k,omega_q)|^2 at the bin of interest
// (PAPER.md:99).  When the modulation frequency is not known, every bin q_lo..q_hi of the N-frame window (nu = q/N) is
// demodulated and each pixel keeps the bin with the largest amplitude R_q = |F_q|.
//
// Fast path (frames whose byte size is a multiple of 16): 32 bins per pass over the stack as ONE launch of the tcgen05
// contraction with 256 columns (32 bins x sin, cos x 4 digits of the Q1.30 references), the arg-max fused into its epilogue;
// the digit tiles of all bins are built once, there is no context and no map per pass: N/64 passes, each HBM-bound.
// Fallback (other frame sizes): eight bins per pass through the public C ABI (qld_create .. qld_destroy) plus one small
// kernel that folds a pass's amplitude maps into the running maximum.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include <mutex>

#include "qld.h"
#include "qld_tc.h"

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

constexpr size_t SEARCH_GROUP_BYTES = 64ull << 20;    // digit tiles built at a time by qld_dominant_bin

// the library's own memory pool on the current device (created on first use, kept until exit; nullptr if that fails)
cudaMemPool_t search_pool()
{
    static std::mutex mu;
    static cudaMemPool_t pools[64] = {nullptr};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { (void)cudaGetLastError(); return nullptr; }
    std::lock_guard<std::mutex> lock(mu);
    if (!pools[dev]) {
        cudaMemPoolProps props;
        memset(&props, 0, sizeof props);
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        if (cudaMemPoolCreate(&pool, &props) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
        uint64_t keep = SEARCH_GROUP_BYTES + (1ull << 20);          // what one search takes stays with the pool between calls
        (void)cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        (void)cudaGetLastError();
        pools[dev] = pool;
    }
    return pools[dev];
}

}  // namespace

extern "C" int qld_dominant_bin(const void *frames_device, int32_t dtype, int32_t H, int32_t W, int32_t N, int32_t q_lo, int32_t q_hi,
                                float *amp_max_device, int32_t *bin_device, void *stream)
{
    if (!frames_device || !amp_max_device || !bin_device || H < 1 || W < 1 || N < 3) return QLD_E_INVAL;
    if (q_lo < 1 || q_hi < q_lo || 2 * (int64_t)q_hi >= N) return QLD_E_INVAL;       // 0 < q/N < 1/2 (reading G18)
    cudaStream_t st = stream ? static_cast<cudaStream_t>(stream) : cudaStreamLegacy;
    const int64_t HW = (int64_t)H * W;
    const int bytes = dtype == QLD_U8 ? 1 : 2;
    if (dtype != QLD_U8 && dtype != QLD_U16 && dtype != QLD_U16_BE) return QLD_E_INVAL;
    if ((HW * bytes) % 16 == 0 && (reinterpret_cast<uintptr_t>(frames_device) & 15) == 0 && N <= 65536) {
        // ---- 32 bins per pass on the tensor cores, arg-max in the epilogue
        const int n_bins = q_hi - q_lo + 1, n_pass = (n_bins + 31) / 32;
        size_t pass_bytes = 0;
        (void)qld_tc_spectrum_digit_bytes(N, n_bins, &pass_bytes);
        // the digit tiles are built for a group of passes at a time (at most SEARCH_GROUP_BYTES: a long window would otherwise
        // ask for 4 N^2 bytes at once) and the groups follow each other in stream order through one buffer
        int group = (int)(SEARCH_GROUP_BYTES / pass_bytes);
        group = group < 1 ? 1 : (group > n_pass ? n_pass : group);
        const size_t dig_bytes = (size_t)group * pass_bytes;
        unsigned char *scratch = nullptr;                    // digit tiles + two tile counters
        // stream-ordered allocation from a pool of the library's own (no device-wide synchronisation on either side of the search;
        // the pool keeps its block between calls; the process's default pool is left as it is)
        cudaMemPool_t pool = search_pool();
        if (!pool || cudaMallocFromPoolAsync(reinterpret_cast<void **>(&scratch), dig_bytes + 256, pool, st) != cudaSuccess) {
            (void)cudaGetLastError();
            scratch = nullptr;                               // no memory for the tiles: the eight-bins-per-pass route below needs far less
        }
        if (scratch) {
            int8_t *digits = reinterpret_cast<int8_t *>(scratch);
            unsigned int *counters = reinterpret_cast<unsigned int *>(scratch + dig_bytes);
            int rc = QLD_OK;
            alignas(64) unsigned char tmaps[256];
            int force[3];
            qld_tc_spectrum_shape(force);
            int n_sms = qld_sm_count();
            if (cudaMemsetAsync(counters, 0, 8, st) != cudaSuccess) rc = QLD_E_CUDA;
            if (rc == QLD_OK && qld_tc_encode_tmap(tmaps, frames_device, HW * bytes, N, 32 /* 256 columns */, n_sms, force) != cudaSuccess) rc = QLD_E_CUDA;
            for (int P = 0; rc == QLD_OK && P < n_pass; ++P) {
                if (P % group == 0) {
                    const int bins_here = n_bins - 32 * P < 32 * group ? n_bins - 32 * P : 32 * group;
                    if (qld_launch_spectrum_digits(N, q_lo + 32 * P, bins_here, digits, st) != cudaSuccess) { rc = QLD_E_CUDA; break; }
                }
                TcParams p;
                memset(&p, 0, sizeof p);
                p.HW = HW; p.row_bytes = HW * bytes; p.N = N; p.bytes = bytes; p.big_endian = dtype == QLD_U16_BE;
                p.digits = digits + (size_t)(P % group) * pass_bytes;
                p.tile_counter = counters + (P & 1); p.tile_counter_next = counters + ((P + 1) & 1);
                p.fin.K = 1; p.fin.scale = 1.0;
                p.spec_amp = amp_max_device; p.spec_bin = bin_device;
                p.spec_q0 = q_lo + 32 * P; p.spec_nbins = n_bins - 32 * P < 32 ? n_bins - 32 * P : 32; p.spec_first = P == 0;
                if (qld_launch_demod_tc_spectrum(tmaps, p, n_sms, st) != cudaSuccess) rc = QLD_E_CUDA;
            }
            cudaFreeAsync(scratch, st);
            if (cudaStreamSynchronize(st) != cudaSuccess) rc = QLD_E_CUDA;
            (void)cudaGetLastError();
            return rc;
        }
    }
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

// ---------------------------------------------------------------------------------------------------------------------
// qld_dominant_bin_static: the tensor-core search above for callers that may not allocate device memory.
//
// Who that is: the acquisition loop of a live camera (the paper's real-time thread) must not stall,
// and cudaMalloc / cudaFree take a driver-wide lock and can wait for every stream of the device -- one search between two
// frame batches would hold up the copies; and a process in which another component (a framework's caching allocator, a
// second library) has already claimed all of HBM has nothing left for qld_dominant_bin's pool allocation to succeed.  For
// them the digit tiles and the two tile counters live in the fixed array below instead.  It is part of the library image:
// every GPU on which the library's kernels are loaded holds these QLD_SEARCH_STATIC_BYTES + 256 bytes until the process
// exits, whether or not the entry point is ever called -- hence the modest size.
//
// The array's name means different things on the two sides.  Device code may use `g_search_scratch` directly.  In host
// code the same name is only a handle the runtime knows the array by -- not an address the GPU can use; a kernel handed
// `g_search_scratch` from the host faults, or, on a system where the GPU can read host memory, quietly works on the wrong
// bytes.  The device address comes from cudaGetSymbolAddress, asked once per device with that device current (each device
// has its own copy of the array at its own address), and that pointer is what the kernels receive.
// ---------------------------------------------------------------------------------------------------------------------
namespace {

constexpr size_t SEARCH_STATIC_TAIL = 256;                            // two tile counters, kept on their own 256 bytes
static __device__ __align__(256) unsigned char g_search_scratch[QLD_SEARCH_STATIC_BYTES + SEARCH_STATIC_TAIL];

constexpr int SEARCH_MAX_DEVICES = 64;
std::mutex g_search_mu;                                               // guards the table below, not the array's contents
unsigned char *g_search_scratch_dev[SEARCH_MAX_DEVICES] = {nullptr};  // device address of the array, per device ordinal
thread_local char g_search_error[256] = "";

int search_fail(int rc, const char *fmt, long long a = 0, long long b = 0)
{
    snprintf(g_search_error, sizeof g_search_error, fmt, a, b);
    return rc;
}

// device address of g_search_scratch on the current device; the first call on a device asks the runtime for it (this
// also makes the runtime load the library's kernels onto that device if nothing did so before)
int search_scratch_address(unsigned char **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        snprintf(g_search_error, sizeof g_search_error, "cudaGetDevice: %s", cudaGetErrorString(e));
        return QLD_E_CUDA;
    }
    if (dev < 0 || dev >= SEARCH_MAX_DEVICES) return search_fail(QLD_E_UNSUPPORTED, "device ordinal %lld is beyond the %lld this entry point keeps addresses for", dev, SEARCH_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_search_mu);
    if (!g_search_scratch_dev[dev]) {
        void *ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_search_scratch);
        if (e != cudaSuccess || !ptr) {
            (void)cudaGetLastError();
            snprintf(g_search_error, sizeof g_search_error, "cudaGetSymbolAddress(g_search_scratch) on device %d: %s", dev, cudaGetErrorString(e));
            return QLD_E_CUDA;
        }
        g_search_scratch_dev[dev] = static_cast<unsigned char *>(ptr);
    }
    *out = g_search_scratch_dev[dev];
    return QLD_OK;
}

}  // namespace

extern "C" const char *qld_dominant_bin_static_error(void) { return g_search_error; }

extern "C" int64_t qld_dominant_bin_static_bytes(int32_t N, int32_t q_lo, int32_t q_hi)
{
    if (N < 3 || q_lo < 1 || q_hi < q_lo || 2 * (int64_t)q_hi >= N || N > 65536) return QLD_E_INVAL;
    return (int64_t)qld_tc_spectrum_digit_bytes(N, q_hi - q_lo + 1, nullptr);
}

extern "C" int qld_dominant_bin_static(const void *frames_device, int32_t dtype, int32_t H, int32_t W, int32_t N, int32_t q_lo, int32_t q_hi,
                                       float *amp_max_device, int32_t *bin_device, void *stream)
{
    g_search_error[0] = 0;
    if (!frames_device || !amp_max_device || !bin_device || H < 1 || W < 1 || N < 3) return search_fail(QLD_E_INVAL, "null pointer, or H, W < 1, or N < 3");
    if (q_lo < 1 || q_hi < q_lo || 2 * (int64_t)q_hi >= N) return search_fail(QLD_E_INVAL, "bins must satisfy 1 <= q_lo <= q_hi and 2 q_hi < N (got %lld..%lld)", q_lo, q_hi);
    if (dtype != QLD_U8 && dtype != QLD_U16 && dtype != QLD_U16_BE) return search_fail(QLD_E_INVAL, "dtype %lld is not a qld_dtype", dtype);
    const int64_t HW = (int64_t)H * W;
    const int bytes = dtype == QLD_U8 ? 1 : 2;
    // only the tensor-core route exists here: qld_dominant_bin's fallback for other frame sizes creates contexts, which allocate
    if ((HW * bytes) % 16 != 0 || (reinterpret_cast<uintptr_t>(frames_device) & 15) != 0 || N > 65536)
        return search_fail(QLD_E_UNSUPPORTED, "needs a 16-byte aligned stack whose frames are a multiple of 16 bytes (frame: %lld bytes) and N <= 65536 (N = %lld)", HW * bytes, N);
    const int n_bins = q_hi - q_lo + 1;
    size_t pass_bytes = 0;
    const size_t dig_bytes = qld_tc_spectrum_digit_bytes(N, n_bins, &pass_bytes);
    if (dig_bytes > (size_t)QLD_SEARCH_STATIC_BYTES)
        return search_fail(QLD_E_NOMEM, "this search needs %lld bytes of digit tiles, the static scratch holds QLD_SEARCH_STATIC_BYTES = %lld: search fewer bins per call or use qld_dominant_bin",
                           (long long)dig_bytes, (long long)QLD_SEARCH_STATIC_BYTES);
    unsigned char *scratch = nullptr;
    int rc = search_scratch_address(&scratch);
    if (rc != QLD_OK) return rc;
    cudaStream_t st = stream ? static_cast<cudaStream_t>(stream) : cudaStreamLegacy;
    int8_t *digits = reinterpret_cast<int8_t *>(scratch);
    unsigned int *counters = reinterpret_cast<unsigned int *>(scratch + QLD_SEARCH_STATIC_BYTES);
    alignas(64) unsigned char tmaps[256];
    int force[3];
    qld_tc_spectrum_shape(force);
    const int n_sms = qld_sm_count();
    cudaError_t e = cudaSuccess;
    const char *where = "";
    // the array still holds the previous call's digits and counters: the counters must start at zero (the tile scheduler counts
    // up from them), the digits this search reads are all rewritten by k_spectrum_digits (padding included) before any pass reads them
    if ((e = cudaMemsetAsync(counters, 0, 8, st)) != cudaSuccess) where = "cudaMemsetAsync(counters)";
    if (e == cudaSuccess && (e = qld_launch_spectrum_digits(N, q_lo, n_bins, digits, st)) != cudaSuccess) where = "k_spectrum_digits";
    if (e == cudaSuccess && (e = qld_tc_encode_tmap(tmaps, frames_device, HW * bytes, N, 32 /* 256 columns */, n_sms, force)) != cudaSuccess) where = "cuTensorMapEncodeTiled";
    for (int P = 0; e == cudaSuccess && P * 32 < n_bins; ++P) {
        TcParams p;
        memset(&p, 0, sizeof p);
        p.HW = HW; p.row_bytes = HW * bytes; p.N = N; p.bytes = bytes; p.big_endian = dtype == QLD_U16_BE;
        p.digits = digits + (size_t)P * pass_bytes;
        p.tile_counter = counters + (P & 1); p.tile_counter_next = counters + ((P + 1) & 1);
        p.fin.K = 1; p.fin.scale = 1.0;
        p.spec_amp = amp_max_device; p.spec_bin = bin_device;
        p.spec_q0 = q_lo + 32 * P; p.spec_nbins = n_bins - 32 * P < 32 ? n_bins - 32 * P : 32; p.spec_first = P == 0;
        if ((e = qld_launch_demod_tc_spectrum(tmaps, p, n_sms, st)) != cudaSuccess) where = "k_demod_tc";
    }
    if (e == cudaSuccess && (e = cudaStreamSynchronize(st)) != cudaSuccess) where = "cudaStreamSynchronize";
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        snprintf(g_search_error, sizeof g_search_error, "%s: %s", where, cudaGetErrorString(e));
        return QLD_E_CUDA;
    }
    return QLD_OK;
}

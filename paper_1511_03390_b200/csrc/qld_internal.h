// Internal declarations shared by the translation units of libqld.so (product side only).
#pragma once
#include <cuda_runtime.h>
#include <atomic>
#include <stdint.h>

#include "qld.h"

#define QLD_MAX_K 8
#define QLD_MAX_ROWS 16

// How one reference maps onto rows of the weight table.
//  FP32     : 2 rows (sin, cos), float weights.
//  INT_BINS : n_rows rows of int weights in {0, +1, -1}; I = sum_r row_r * sw[r], Q = sum_r row_r * cw[r].
struct RefPlan {
    double nu, phase;
    int64_t num, den;
    int32_t phase_quarter;
    int32_t row_off, n_rows;
    int32_t use_diff;  // 1: even den, rows are B_r - B_{r+den/2};  0: rows are the bins B_r;  2: integer-valued scaled references
                       // (den = 3 or 6, no phase): row 0 = sum x * (2/sqrt3) sin theta_s, row 1 = sum x * 2 cos theta_s, weights in 0, +-1, +-2
};

// Epilogue (A4) parameters, passed by value to the kernels.
struct FinParams {
    int32_t K;
    int32_t is_int;          // 1: rows are int32 bins, combine with sw/cw;  0: row_off = I sum, row_off+1 = Q sum
    int32_t row_off[QLD_MAX_K];
    int32_t n_rows[QLD_MAX_K];
    double sw[QLD_MAX_ROWS]; // per row: sin(2 pi r/den + phase)
    double cw[QLD_MAX_ROWS];
    double scale;            // 1 (PAPER) or 2/N (AMPLITUDE)
    float *I, *Q, *amp, *phase;   // [K][HW] or null
    const double *rot;       // window-relative I/Q (reading G10): device array {cos d_k, sin d_k}, d_k = 2 pi nu_k (frames before
                             // the window); null: references by absolute frame index only
};

// A run of consecutive store slots (no wrap inside a run) whose frames enter the sums with weight sign * w:
// a whole window is one or two runs with sign +1 (a ring wraps once); a sliding update (A5) is the expired
// frames with sign -1 followed by the new frames with sign +1.  k_demod_stream walks runs; k_demod_whole uses
// slot0 / n / w0.
struct DemodRun {
    int32_t slot0, n;        // first slot, number of frames
    int32_t w0;              // weight entry of the first frame (entries wrap at cap_w)
    int32_t sign;            // +1 or -1
};

// One demodulation launch (whole window, ring aware).
struct DemodParams {
    const void *frames;      // frame store base
    int64_t frame_stride;    // bytes between frames
    int64_t HW;
    int32_t cap;             // frame store capacity (frames); slot of frame s is (s-1) mod cap
    int32_t slot0;           // slot of the first frame of the window
    int32_t n;               // frames in the window
    int32_t cap_w;           // weight table capacity; entry of frame s is s mod cap_w
    int32_t w0;              // weight entry of the first frame
    int32_t cum_lo, cum_hi;  // weight entries of frame (first-1) and of the last frame, for the pedestal sums
    const void *wtab;        // [cap_w][ROWS] float or int32
    const double *cum;       // [cap_w][ROWS] running sums of the float weights (FP32 only)
    void *acc_out;           // optional [ROWS][HW]: double (FP32: pedestal-subtracted sums) or int32 (bins)
    float *ped_out;          // optional [HW] pedestal used (FP32)
    // k_demod_stream only
    int32_t n_runs;
    int32_t onehot;          // integer bins, one reference: every weight row is one-hot (+-1 in one row)
    int32_t acc_add;         // 1: acc_out holds the previous window's sums; this launch's sums are added to them
    DemodRun run[4];
    void *part;              // block-partial sliding (8(f3)): [ROWS][HW] slot of the partial-sum ring; this launch's sums are
                             // stored there, after the slot's previous content was taken off acc_out when part_sub is set
    int32_t part_sub;
    int32_t big_endian;      // 16-bit samples arrive most significant byte first (QLD_U16_BE): stitched in the load
    const float *ped_in;     // FP32: pedestal to subtract (the one acc_out was seeded with); NULL: the first sample
    FinParams fin;
};

// One sliding update launch (A5).
struct SlideParams {
    const void *frames;
    int64_t frame_stride;
    int64_t HW;
    int32_t cap, cap_w;
    int32_t new_slot0, old_slot0;   // slots of the first new / first expired frame
    int32_t new_w0, old_w0;         // weight entries of the same
    int32_t hop;
    int32_t big_endian;
    int32_t cum_lo, cum_hi;         // entries of frame (window first - 1) and window last, after the update
    const void *wtab;
    const double *cum;
    void *acc;                      // [ROWS][HW] double or int32, read-modify-write
    const float *ped;               // [HW] (FP32)
    FinParams fin;
};

struct TableFillParams {
    int32_t K, is_int, rows;        // is_int: 0 float rows, 1 integer bin indicators, 2 Q1.30 integers; rows = padded row count (row stride)
    RefPlan ref[QLD_MAX_K];
    int64_t s_first;
    int32_t n, cap_w;
    void *wtab;
    double *cum;
};

// launchers (return cudaError_t of the launch)
cudaError_t qld_launch_demod_whole(int dtype, int is_int, int rows, const DemodParams &p, cudaStream_t st);
cudaError_t qld_launch_demod_slide(int dtype, int is_int, int rows, const SlideParams &p, cudaStream_t st);
cudaError_t qld_launch_table_fill(const TableFillParams &p, cudaStream_t st);
// rows (row0, row0 + 1) of the float table from caller-supplied doubles tab[2][n] (sin, cos), frames 1..n; recomputes cum
cudaError_t qld_launch_table_from_doubles(const double *tab, int n, int row0, int rows, int cap_w, void *wtab, double *cum, cudaStream_t st);
// rot[2k], rot[2k+1] = cos, sin of 2 pi nu_k a (a = frames before the window), exactly reduced
cudaError_t qld_launch_window_rotation(const TableFillParams &p, int64_t a, double *rot, cudaStream_t st);
cudaError_t qld_launch_bin_weights(const TableFillParams &p, double *out32 /* device: sw[16], cw[16] */, cudaStream_t st);
int qld_pixels_per_thread(int dtype, int rows, int64_t HW, const void *frames, int64_t frame_stride);

// multiprocessor count of the current device (cached per device)
inline int qld_sm_count()
{
    static int cached[64] = {0};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 1;
    int &n = cached[dev & 63];
    if (n == 0 && cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) n = 1;
    return n > 0 ? n : 1;
}

// Lift a kernel's dynamic shared-memory limit to the device's opt-in maximum, once per (kernel instantiation, device);
// `done` is the instantiation's own zero-initialised table.  Whoever writes the attribute writes the same value, so two host
// threads that launch different tile shapes of one kernel at the same time (distinct contexts are independent across threads,
// qld.h) cannot leave it below what a later launch needs -- which a cached "largest size set so far" could.
template <typename Kernel>
inline cudaError_t qld_allow_max_smem(Kernel kern, std::atomic<int> (&done)[64])
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool cached = dev >= 0 && dev < 64;
    if (cached && done[dev].load(std::memory_order_acquire)) return cudaSuccess;
    int optin = 0;
    e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    if (e != cudaSuccess) return e;
    if (cached) done[dev].store(1, std::memory_order_release);
    return cudaSuccess;
}

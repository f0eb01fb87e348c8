// A1: reference tables ("pre-calculated arrays"; "tables of sine and cosine functions,
// appropriate for the choice of lock-in and sampling frequencies"), filled on the device.
//
// theta_{k,s} = 2*pi*nu_k*s + phase_k, s = absolute frame index starting at 1.  The turn count
// nu*s is reduced modulo 1 *before* any trigonometry: exactly in integers for rational nu = num/den, and with
// an fma-recovered exact product for real nu, then fp64 sincospi, rounded once to fp32.  The same entry is
// used when a frame enters a sliding window and when it leaves it.
// For INT_BINS the rows are integer indicators of the phase bin r = num*s mod den (see include/qld.h).
// A running fp64 sum of every float row (cum) provides sum_s w(s) over any window for the pedestal term.
#include "qld_internal.h"

namespace {

__device__ __forceinline__ int64_t bin_of(const RefPlan &rf, int64_t s)
{
    const uint64_t a = (uint64_t)(rf.num % rf.den), b = (uint64_t)(s % rf.den);
    return (int64_t)((a * b) % (uint64_t)rf.den);      // den < 2^31: the product fits 64 bits
}

__device__ __forceinline__ double half_turns_of(const RefPlan &rf, int64_t s)
{
    double a;
    if (rf.den > 0) {
        a = 2.0 * (double)bin_of(rf, s) / (double)rf.den;
    } else {
        const double sd = (double)s;
        const double hi = rf.nu * sd;
        const double lo = fma(rf.nu, sd, -hi);          // exact low part of nu*s
        a = 2.0 * ((hi - floor(hi)) + lo);
    }
    a += 0.5 * (double)(rf.phase_quarter & 3);
    if (rf.phase != 0.0) a += rf.phase * 0.31830988618379067154;   // phase / pi
    return a;
}

__global__ void k_table_fill(const TableFillParams p)
{
    for (int idx = threadIdx.x; idx < p.n * p.K; idx += blockDim.x) {
        const int i = idx / p.K, k = idx % p.K;
        const RefPlan &rf = p.ref[k];
        const int64_t s = p.s_first + i;
        const int64_t e = s % p.cap_w;
        if (!p.is_int) {
            double sn, cs;
            sincospi(half_turns_of(rf, s), &sn, &cs);
            float *w = static_cast<float *>(p.wtab) + e * p.rows + rf.row_off;
            w[0] = (float)sn;
            w[1] = (float)cs;
        } else {
            const int64_t r = bin_of(rf, s);
            int *w = static_cast<int *>(p.wtab) + e * p.rows + rf.row_off;
            const int64_t half = rf.den / 2;
            for (int rr = 0; rr < rf.n_rows; ++rr)
                w[rr] = rf.use_diff ? ((r == rr) - (r == rr + half)) : (r == rr);
        }
    }
    __syncthreads();
    if (!p.is_int) {
        for (int r = threadIdx.x; r < p.rows; r += blockDim.x) {
            const float *w = static_cast<const float *>(p.wtab);
            double c = p.cum[((p.s_first - 1) % p.cap_w) * p.rows + r];
            for (int i = 0; i < p.n; ++i) {
                const int64_t e = (p.s_first + i) % p.cap_w;
                c += (double)w[e * p.rows + r];
                p.cum[e * p.rows + r] = c;
            }
        }
    }
}

}  // namespace

cudaError_t qld_launch_table_fill(const TableFillParams &p, cudaStream_t st)
{
    k_table_fill<<<1, 256, 0, st>>>(p);
    return cudaGetLastError();
}

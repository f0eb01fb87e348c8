// A1: reference tables ("pre-calculated arrays"; "tables of sine and cosine functions,
// appropriate for the choice of lock-in and sampling frequencies"), filled on the device.
//
// theta_{k,s} = 2*pi*nu_k*s + phase_k, s = absolute frame index starting at 1.  The turn count
// nu*s is reduced modulo 1 *before* any trigonometry: exactly in integers for rational nu = num/den, and with
// an fma-recovered exact product for real nu, then fp64 sincospi, rounded once to fp32.  The same entry is
// used when a frame enters a sliding window and when it leaves it.
// For INT_BINS the rows are integer indicators of the phase bin r = num*s mod den (see include/qld.h).
// A running fp64 sum of every float row (cum) provides sum_s w(s) over any window for the pedestal term.
#include "qld_angle.cuh"
#include "qld_internal.h"

using namespace qld_angle;

namespace {

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
        } else if (p.is_int == 2) {
            // Q1.30 fixed-point references (drift-free sliding at any nu): rint(2^30 sin), rint(2^30 cos)
            double sn, cs;
            sincospi(half_turns_of(rf, s), &sn, &cs);
            int *w = static_cast<int *>(p.wtab) + e * p.rows + rf.row_off;
            w[0] = (int)rint(sn * 1073741824.0);
            w[1] = (int)rint(cs * 1073741824.0);
        } else {
            const int64_t r = bin_of(rf, s);
            int *w = static_cast<int *>(p.wtab) + e * p.rows + rf.row_off;
            const int64_t half = rf.den / 2;
            if (rf.use_diff == 2) {
                // theta = 2 pi r / den with den = 3 or 6: (2/sqrt3) sin theta and 2 cos theta are the integers below (sixths of a turn)
                const int wi6[6] = {0, 1, 1, 0, -1, -1}, wq6[6] = {2, 1, -1, -2, -1, 1};
                const int j = (int)(rf.den == 6 ? r : 2 * r);
                w[0] = wi6[j];
                w[1] = wq6[j];
            } else {
                for (int rr = 0; rr < rf.n_rows; ++rr)
                    w[rr] = rf.use_diff ? ((r == rr) - (r == rr + half)) : (r == rr);
            }
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

// INT_BINS combine weights: row r of reference k holds the (difference of) phase-bin sums whose frames all carry the
// reference value sin / cos(2*pi*r/den + phase), so I = sum_r row_r * sw[r], Q = sum_r row_r * cw[r] (include/qld.h).
// With no free phase the angle is the rational a/D of a turn, D = 4*den, a = 4*r + phase_quarter*den; whenever that is a
// whole number j of twelfths of a turn the value is taken from the twelve-entry table of 2*sin(j*30 deg) =
// 0, 1, sqrt3, 2, sqrt3, 1, 0, -1, ... halved (exact 0, +-1/2, +-1; sqrt3/2 correctly rounded) -- this is what makes
// nu = 1/4 integer valued and nu = 1/6 exact in its halves; every other angle goes through fp64 sincospi of the reduced
// half-turn count.  out[0..15] = sw, out[16..31] = cw (zeros for padding rows).
__global__ void k_bin_weights(const TableFillParams p, double *out)
{
    const int t = threadIdx.x;
    if (t >= 2 * QLD_MAX_ROWS) return;
    out[t] = 0.0;
    if (t >= QLD_MAX_ROWS) return;
    for (int k = 0; k < p.K; ++k) {
        const RefPlan &rf = p.ref[k];
        const int r = t - rf.row_off;
        if (r < 0 || r >= rf.n_rows) continue;
        if (rf.use_diff == 2) {
            // scaled integer references: I = (sqrt3 / 2) * row 0, Q = (1/2) * row 1
            out[t] = r == 0 ? 0.5 * sqrt(3.0) : 0.0;
            out[QLD_MAX_ROWS + t] = r == 1 ? 0.5 : 0.0;
            continue;
        }
        const int64_t D = 4 * rf.den;
        const int64_t a = (4 * (int64_t)r + (int64_t)(rf.phase_quarter & 3) * rf.den) % D;
        double sn, cs;
        if (rf.phase == 0.0 && (12 * a) % D == 0) {
            const double r3 = sqrt(3.0);
            const double twice_sin[12] = {0.0, 1.0, r3, 2.0, r3, 1.0, 0.0, -1.0, -r3, -2.0, -r3, -1.0};
            const int j = (int)((12 * a) / D);
            sn = 0.5 * twice_sin[j];
            cs = 0.5 * twice_sin[(j + 3) % 12];           // cos x = sin(x + 90 deg)
        } else {
            sincospi(2.0 * (double)a / (double)D + rf.phase * 0.31830988618379067154, &sn, &cs);
        }
        out[t] = sn;
        out[QLD_MAX_ROWS + t] = cs;
    }
}

// caller-supplied tables (qld_set_ref_tables): rounded once to fp32, running sums redone for the two rows
__global__ void k_table_from_doubles(const double *tab, int n, int row0, int rows, int cap_w, float *wtab, double *cum)
{
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const int64_t e = (int64_t)(i + 1) % cap_w;
        wtab[e * rows + row0] = (float)tab[i];
        wtab[e * rows + row0 + 1] = (float)tab[n + i];
    }
    __syncthreads();
    if (threadIdx.x < 2) {
        const int r = row0 + threadIdx.x;
        double c = 0.0;                                   // entry of frame 0
        cum[r] = 0.0;
        for (int i = 0; i < n; ++i) {
            const int64_t e = (int64_t)(i + 1) % cap_w;
            c += (double)wtab[e * rows + r];
            cum[e * rows + r] = c;
        }
    }
}

// Window-relative I / Q (reading G10): a window that starts after `a` frames sees references that are
// d = 2 pi nu a ahead of window-relative ones; the epilogues turn (I, Q) back by d.  rot = {cos d, sin d} per reference.
__global__ void k_window_rotation(const TableFillParams p, int64_t a, double *rot)
{
    const int k = threadIdx.x;
    if (k >= p.K) return;
    RefPlan rf = p.ref[k];
    rf.phase = 0.0;
    rf.phase_quarter = 0;
    double sn, cs;
    sincospi(half_turns_of(rf, a), &sn, &cs);
    rot[2 * k] = cs;
    rot[2 * k + 1] = sn;
}

}  // namespace

cudaError_t qld_launch_window_rotation(const TableFillParams &p, int64_t a, double *rot, cudaStream_t st)
{
    k_window_rotation<<<1, 32, 0, st>>>(p, a, rot);
    return cudaGetLastError();
}

cudaError_t qld_launch_table_from_doubles(const double *tab, int n, int row0, int rows, int cap_w, void *wtab, double *cum, cudaStream_t st)
{
    k_table_from_doubles<<<1, 256, 0, st>>>(tab, n, row0, rows, cap_w, static_cast<float *>(wtab), cum);
    return cudaGetLastError();
}

cudaError_t qld_launch_bin_weights(const TableFillParams &p, double *out32, cudaStream_t st)
{
    k_bin_weights<<<1, 2 * QLD_MAX_ROWS, 0, st>>>(p, out32);
    return cudaGetLastError();
}

cudaError_t qld_launch_table_fill(const TableFillParams &p, cudaStream_t st)
{
    k_table_fill<<<1, 256, 0, st>>>(p);
    return cudaGetLastError();
}

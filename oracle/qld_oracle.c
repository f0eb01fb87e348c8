/*
 * qld_oracle.c -- CPU oracle for quadrature lock-in discrimination (QLD), arXiv 1511.03390.
 *
 * TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * `--impl reference` legs may build, load or call this file.  The product (the CUDA library
 * behind include/qld.h) shares no code, header, table or helper with it and never calls it.
 *
 * What it computes is the paper's definition, written out plainly (DESIGN.md "Readings" G1-G7):
 *
 *   PAPER.md:99 (Methods):  R(j,k) = [ (sum_s I(j,k,t_s) sin(w t_s))^2 + (sum_s I(j,k,t_s) cos(w t_s))^2 ]^(1/2)
 *                           with sin/cos "read from pre-calculated arrays";
 *   PAPER.md:97:            t_s = s*dt, s = 1, 2, ... N   (frame index starts at 1);
 *   PAPER.md:169:           per frame, intensity * sin and intensity * cos are accumulated into two
 *                           2-D arrays (the two quadrature components), then squared and added;
 *   PAPER.md:31:            one copy is multiplied by the reference sinusoid (in-phase, "I" = sin sum),
 *                           the other by the 90-degree shifted one (quadrature, "Q" = cos sum).
 *
 * The extracted formula at PAPER.md:99 has the squares inside the sums; that literal form equals
 * sum_s I^2 and cannot discriminate a frequency, and PAPER.md:169 says accumulate first, square
 * after -- so the sums are squared (reading G1).  No normalisation, no mean removal (G3, G9).
 *
 * Arithmetic: samples are integers converted exactly; float paths accumulate in x87 `long double`
 * (64-bit significand) in frame order, the streaming order of PAPER.md:169, and round once to
 * double at the end; integer paths use int64_t throughout.  There is no blocking, no reordering
 * and no fusion beyond that.  OpenMP, when nthreads > 1, only splits the *pixel* range between
 * threads ("multi-CPU"); each pixel's sum is still sequential in s.
 *
 * Pins: tests/test_oracle_pins.py (closed forms, DFT bins via numpy.fft, Parseval, brute force in
 * Python integers, mpmath angles).  Nothing here is "parity unpinned" except the paper's CNR
 * figures, which are outside this file (inputs not reproducible).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define QLDO_U8 0
#define QLDO_U16 1
#define QLDO_F64 2

static const long double TWO_PI_L = 6.283185307179586476925286766559005768L;

/* ------------------------------------------------------------------------------------------
 * Reference tables ("pre-calculated arrays", "tables of sine and cosine
 * functions, appropriate for the choice of lock-in and sampling frequencies").
 * theta_s = 2*pi*nu*s + phase, nu = f_mod/f_s (dimensionless; the paper gives Hz without dt, G8).
 * ---------------------------------------------------------------------------------------- */

/* Real nu: the turn count nu*s is reduced modulo 1 before multiplying by 2*pi, with the exact
 * product recovered by fmal, so large s does not lose the angle. */
void qldo_ref_real(double nu, double phase, int64_t s_first, int64_t n, double *sin_tab, double *cos_tab)
{
    for (int64_t i = 0; i < n; ++i) {
        long double s = (long double)(s_first + i);
        long double hi = (long double)nu * s;
        long double lo = fmal((long double)nu, s, -hi);   /* exact low part of nu*s */
        long double fr = (hi - floorl(hi)) + lo;
        long double th = TWO_PI_L * fr + (long double)phase;
        sin_tab[i] = (double)sinl(th);
        cos_tab[i] = (double)cosl(th);
    }
}

/* Rational nu = num/den, reference phase = phase_quarter*(pi/2) + phase.  The turn fraction
 * (num*s mod den)/den + phase_quarter/4 is kept as an exact rational a/D; multiples of a quarter
 * turn give exactly 0, +-1 and multiples of a twelfth give exactly +-1/2 (libm would return
 * sin(pi) = 1.2e-16 and sin(pi/6) = 0.49999999999999994), which is what makes the nu = 1/4
 * table integer valued. */
static void exact_sincos_turn(int64_t a, int64_t D, long double extra, double *sn, double *cs)
{
    static const int q_sin[4] = {0, 1, 0, -1};
    static const int q_cos[4] = {1, 0, -1, 0};
    if (extra == 0.0L && (4 * a) % D == 0) {
        int j = (int)((4 * a) / D) & 3;
        *sn = q_sin[j];
        *cs = q_cos[j];
        return;
    }
    long double th = TWO_PI_L * ((long double)a / (long double)D) + extra;
    long double s = sinl(th), c = cosl(th);
    if (extra == 0.0L && (12 * a) % D == 0) {
        int j = (int)((12 * a) / D) % 12;               /* angle = j * 30 degrees */
        if (j == 1 || j == 5) s = 0.5L;
        if (j == 7 || j == 11) s = -0.5L;
        if (j == 2 || j == 10) c = 0.5L;
        if (j == 4 || j == 8) c = -0.5L;
    }
    *sn = (double)s;
    *cs = (double)c;
}

void qldo_ref_rational(int64_t num, int64_t den, int64_t phase_quarter, double phase, int64_t s_first, int64_t n,
                       double *sin_tab, double *cos_tab)
{
    int64_t D = 4 * den;
    int64_t pq = ((phase_quarter % 4) + 4) % 4;
    for (int64_t i = 0; i < n; ++i) {
        int64_t s = s_first + i;
        int64_t r = (int64_t)((((__int128)(num % den)) * (__int128)(((s % den) + den) % den)) % den);
        if (r < 0) r += den;
        int64_t a = (4 * r + pq * den) % D;
        exact_sincos_turn(a, D, (long double)phase, &sin_tab[i], &cos_tab[i]);
    }
}

/* Phase-bin index of frame s for nu = num/den: r = (num * s) mod den, so theta_s = 2*pi*r/den. */
void qldo_bin_index(int64_t num, int64_t den, int64_t s_first, int64_t n, int32_t *bin)
{
    for (int64_t i = 0; i < n; ++i) {
        int64_t s = s_first + i;
        int64_t r = (int64_t)((((__int128)(num % den)) * (__int128)(((s % den) + den) % den)) % den);
        if (r < 0) r += den;
        bin[i] = (int32_t)r;
    }
}

/* ------------------------------------------------------------------------------------------
 * The sums.  frames: [n_frames][hw] row-major (frame-major, pixels contiguous), dtype as given.
 * ---------------------------------------------------------------------------------------- */
static inline long double sample_ld(const void *frames, int dtype, int64_t idx)
{
    switch (dtype) {
    case QLDO_U8: return (long double)((const uint8_t *)frames)[idx];
    case QLDO_U16: return (long double)((const uint16_t *)frames)[idx];
    default: return (long double)((const double *)frames)[idx];
    }
}

static inline int64_t sample_i64(const void *frames, int dtype, int64_t idx)
{
    return dtype == QLDO_U8 ? (int64_t)((const uint8_t *)frames)[idx] : (int64_t)((const uint16_t *)frames)[idx];
}

/* S(p) = sum_s x_s(p) sin_tab[s],  C(p) = sum_s x_s(p) cos_tab[s].
 * pix_stride lets a caller pass a sub-range of pixels of a larger frame: frame f starts at
 * frames + f*frame_stride (in samples).  Returns 0, or -1 on a bad dtype. */
int qldo_demod_f64(const void *frames, int dtype, int64_t n_frames, int64_t hw, int64_t frame_stride,
                   const double *sin_tab, const double *cos_tab, double *S, double *C, int nthreads)
{
    if (dtype < 0 || dtype > 2) return -1;
    if (nthreads < 1) nthreads = 1;
    int64_t chunk = (hw + nthreads - 1) / nthreads;
#pragma omp parallel for num_threads(nthreads) schedule(static)
    for (int t = 0; t < nthreads; ++t) {
        int64_t p0 = (int64_t)t * chunk, p1 = p0 + chunk < hw ? p0 + chunk : hw;
        if (p0 >= p1) continue;
        int64_t m = p1 - p0;
        long double *accS = (long double *)calloc((size_t)m, sizeof(long double));
        long double *accC = (long double *)calloc((size_t)m, sizeof(long double));
        for (int64_t s = 0; s < n_frames; ++s) {            /* frame order: s = 1 .. N */
            long double sn = (long double)sin_tab[s], cs = (long double)cos_tab[s];
            for (int64_t p = p0; p < p1; ++p) {
                long double x = sample_ld(frames, dtype, s * frame_stride + p);
                accS[p - p0] += x * sn;                     /* intermediate "sin frame", accumulated */
                accC[p - p0] += x * cs;                     /* intermediate "cos frame", accumulated */
            }
        }
        for (int64_t p = p0; p < p1; ++p) {
            S[p] = (double)accS[p - p0];
            C[p] = (double)accC[p - p0];
        }
        free(accS);
        free(accC);
    }
    return 0;
}

/* Integer-valued references (e.g. nu = 1/4, phase a multiple of pi/2: table in {0, +-1}; or
 * fixed-point references): the same sums in exact int64 arithmetic. */
int qldo_demod_i64(const void *frames, int dtype, int64_t n_frames, int64_t hw, int64_t frame_stride,
                   const int64_t *isin, const int64_t *icos, int64_t *S, int64_t *C, int nthreads)
{
    if (dtype != QLDO_U8 && dtype != QLDO_U16) return -1;
    if (nthreads < 1) nthreads = 1;
    int64_t chunk = (hw + nthreads - 1) / nthreads;
#pragma omp parallel for num_threads(nthreads) schedule(static)
    for (int t = 0; t < nthreads; ++t) {
        int64_t p0 = (int64_t)t * chunk, p1 = p0 + chunk < hw ? p0 + chunk : hw;
        for (int64_t p = p0; p < p1; ++p) { S[p] = 0; C[p] = 0; }
        for (int64_t s = 0; s < n_frames; ++s)
            for (int64_t p = p0; p < p1; ++p) {
                int64_t x = sample_i64(frames, dtype, s * frame_stride + p);
                S[p] += x * isin[s];
                C[p] += x * icos[s];
            }
    }
    return 0;
}

/* Phase-bin sums for nu = num/den: B[r][p] = sum over frames s with bin[s] == r of x_s(p).
 * Then S = sum_r B_r sin(2 pi r/den + phi), C likewise -- the same sums as qldo_demod_f64 with the
 * terms grouped by equal reference value (exact regrouping: within a bin the reference is one
 * constant).  B: [den][hw] int64. */
int qldo_bins_i64(const void *frames, int dtype, int64_t n_frames, int64_t hw, int64_t frame_stride,
                  const int32_t *bin, int64_t den, int64_t *B)
{
    if (dtype != QLDO_U8 && dtype != QLDO_U16) return -1;
    memset(B, 0, (size_t)(den * hw) * sizeof(int64_t));
    for (int64_t s = 0; s < n_frames; ++s) {
        int64_t *row = B + (int64_t)bin[s] * hw;
        for (int64_t p = 0; p < hw; ++p) row[p] += sample_i64(frames, dtype, s * frame_stride + p);
    }
    return 0;
}

/* Amplitude R = sqrt(S^2 + C^2) (exponent 1/2) and phase = atan2(C, S), 0 when
 * S = C = 0 (the paper has no phase map; BASELINE.json asks for one; reading G6: a source
 * A sin(theta_s + phi) gives S = (AN/2) cos phi, C = (AN/2) sin phi, so atan2(C, S) = phi). */
void qldo_finalise(const double *S, const double *C, int64_t hw, double scale, double *R, double *phase)
{
    for (int64_t p = 0; p < hw; ++p) {
        long double s = (long double)S[p] * scale, c = (long double)C[p] * scale;
        if (R) R[p] = (double)sqrtl(s * s + c * c);
        if (phase) phase[p] = (S[p] == 0.0 && C[p] == 0.0) ? 0.0 : (double)atan2l(c, s);
    }
}

int qldo_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// Reference angles on the device (A1; "pre-calculated arrays"): shared by the table kernels of
// qld_tables.cu (fp32 / bin-weight tables) and qld_tc.cu (Q1.30 fixed-point tables).
//
// theta_{k,s} = 2*pi*nu_k*s + phase_k with s the absolute frame index from 1.  The turn count nu*s is reduced
// modulo 1 before any trigonometry -- exactly in integers for rational nu = num/den, with an fma-recovered exact product for
// real nu -- and the result is handed to fp64 sincospi as a number of half turns.
#pragma once
#include "qld_internal.h"

namespace qld_angle {

// phase bin of frame s for nu = num/den: r = num*s mod den, so that theta_s = 2*pi*r/den (+ phase)
__device__ __forceinline__ int64_t bin_of(const RefPlan &rf, int64_t s)
{
    const uint64_t a = (uint64_t)(rf.num % rf.den), b = (uint64_t)(s % rf.den);
    return (int64_t)((a * b) % (uint64_t)rf.den);      // den < 2^31: the product fits 64 bits
}

// theta_{k,s} / pi, reduced
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

}  // namespace qld_angle

// Device helpers shared by the demodulation kernels (qld_kernels.cu, qld_stream.cu): sample unpacking, the
// per-frame multiply-accumulate ("multiplied by two numbers ... accumulated"), and the A4 epilogue.
#pragma once
#include <type_traits>

#include "qld_internal.h"

namespace qld_dev {

// ---------------------------------------------------------------------------------------------------
// streaming loads of V samples of type T (V * sizeof(T) bytes <= 16)
// ---------------------------------------------------------------------------------------------------
template <typename T, int V>
struct Pix {
    static constexpr int VB = V * (int)sizeof(T);
    static constexpr int NW = (VB + 3) / 4;
    static_assert(VB == 1 || VB == 2 || VB == 4 || VB == 8 || VB == 16, "vector width");

    __device__ __forceinline__ static void load(const unsigned char *ptr, uint32_t (&w)[NW])
    {
        if constexpr (VB == 16) {
            asm("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]) : "l"(ptr));
        } else if constexpr (VB == 8) {
            asm("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(w[0]), "=r"(w[1]) : "l"(ptr));
        } else if constexpr (VB == 4) {
            asm("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(w[0]) : "l"(ptr));
        } else if constexpr (VB == 2) {
            w[0] = *reinterpret_cast<const unsigned short *>(ptr);
        } else {
            w[0] = *ptr;
        }
    }
    // the same V samples from shared memory (TMA-staged tiles)
    __device__ __forceinline__ static void load_shared(const unsigned char *ptr, uint32_t (&w)[NW])
    {
        if constexpr (VB == 16) {
            const uint4 t = *reinterpret_cast<const uint4 *>(ptr);
            w[0] = t.x; w[1] = t.y; w[2] = t.z; w[3] = t.w;
        } else if constexpr (VB == 8) {
            const uint2 t = *reinterpret_cast<const uint2 *>(ptr);
            w[0] = t.x; w[1] = t.y;
        } else if constexpr (VB == 4) {
            w[0] = *reinterpret_cast<const uint32_t *>(ptr);
        } else if constexpr (VB == 2) {
            w[0] = *reinterpret_cast<const unsigned short *>(ptr);
        } else {
            w[0] = *ptr;
        }
    }
    // bsw: selector mask that stitches the byte pair of a 16-bit sample the other way round (QLD_U16_BE, a Camera-Link style
    // stream with the most significant byte first): 0x11 swaps the two low selector nibbles, 0 = little endian
    // sample j as an unsigned integer
    __device__ __forceinline__ static uint32_t geti(const uint32_t (&w)[NW], int j, uint32_t bsw = 0)
    {
        // one byte-permute (selector nibble 4 = a zero byte of the second operand)
        if constexpr (sizeof(T) == 2) return __byte_perm(w[j >> 1], 0u, ((j & 1) ? 0x4432u : 0x4410u) ^ bsw);
        else return __byte_perm(w[j >> 2], 0u, 0x4440u | (uint32_t)(j & 3));
    }
    // sample j as the float 2^23 + x (one byte-permute: the integer lands in the mantissa of 0x4B000000)
    __device__ __forceinline__ static float getf_biased(const uint32_t (&w)[NW], int j, uint32_t bsw = 0)
    {
        uint32_t r;
        if constexpr (sizeof(T) == 2) r = __byte_perm(w[j >> 1], 0x4B000000u, ((j & 1) ? 0x7632u : 0x7610u) ^ bsw);
        else r = __byte_perm(w[j >> 2], 0x4B000000u, 0x7650u | (uint32_t)(j & 3));
        return __uint_as_float(r);
    }
};

// N consecutive values of type E (N * sizeof(E) a multiple of 16, pointer 16-byte aligned) as 16-byte accesses
template <typename E, int N>
__device__ __forceinline__ void load_vec(const E *ptr, E (&out)[N])
{
    constexpr int PER = 16 / (int)sizeof(E);
    if constexpr (N % PER == 0) {
#pragma unroll
        for (int i = 0; i < N / PER; ++i) {
            const int4 t = reinterpret_cast<const int4 *>(ptr)[i];
            alignas(16) E tmp[PER];
            *reinterpret_cast<int4 *>(tmp) = t;
#pragma unroll
            for (int j = 0; j < PER; ++j) out[i * PER + j] = tmp[j];
        }
    } else {
#pragma unroll
        for (int i = 0; i < N; ++i) out[i] = ptr[i];
    }
}
template <typename E, int N>
__device__ __forceinline__ void store_vec(E *ptr, const E (&in)[N])
{
    constexpr int PER = 16 / (int)sizeof(E);
    if constexpr (N % PER == 0) {
#pragma unroll
        for (int i = 0; i < N / PER; ++i) {
            alignas(16) E tmp[PER];
#pragma unroll
            for (int j = 0; j < PER; ++j) tmp[j] = in[i * PER + j];
            reinterpret_cast<int4 *>(ptr)[i] = *reinterpret_cast<const int4 *>(tmp);
        }
    } else {
#pragma unroll
        for (int i = 0; i < N; ++i) ptr[i] = in[i];
    }
}

// weights of one frame: ROWS values, identical for every thread (broadcast load through L1)
template <typename ACC, int ROWS>
__device__ __forceinline__ void load_weights(const ACC *row, ACC (&wt)[ROWS])
{
    if constexpr (ROWS % 4 == 0) {
#pragma unroll
        for (int q = 0; q < ROWS / 4; ++q) {
            int4 t = __ldg(reinterpret_cast<const int4 *>(row) + q);
            wt[4 * q + 0] = *reinterpret_cast<ACC *>(&t.x);
            wt[4 * q + 1] = *reinterpret_cast<ACC *>(&t.y);
            wt[4 * q + 2] = *reinterpret_cast<ACC *>(&t.z);
            wt[4 * q + 3] = *reinterpret_cast<ACC *>(&t.w);
        }
    } else if constexpr (ROWS % 2 == 0) {
#pragma unroll
        for (int q = 0; q < ROWS / 2; ++q) {
            int2 t = __ldg(reinterpret_cast<const int2 *>(row) + q);
            wt[2 * q + 0] = *reinterpret_cast<ACC *>(&t.x);
            wt[2 * q + 1] = *reinterpret_cast<ACC *>(&t.y);
        }
    } else {
#pragma unroll
        for (int q = 0; q < ROWS; ++q) wt[q] = __ldg(row + q);
    }
}

// the same from a shared-memory copy of the rows
template <typename ACC, int ROWS>
__device__ __forceinline__ void load_weights_shared(const ACC *row, ACC (&wt)[ROWS])
{
    if constexpr (ROWS % 4 == 0) {
#pragma unroll
        for (int q = 0; q < ROWS / 4; ++q) {
            const int4 t = reinterpret_cast<const int4 *>(row)[q];
            wt[4 * q + 0] = *reinterpret_cast<const ACC *>(&t.x);
            wt[4 * q + 1] = *reinterpret_cast<const ACC *>(&t.y);
            wt[4 * q + 2] = *reinterpret_cast<const ACC *>(&t.z);
            wt[4 * q + 3] = *reinterpret_cast<const ACC *>(&t.w);
        }
    } else if constexpr (ROWS % 2 == 0) {
#pragma unroll
        for (int q = 0; q < ROWS / 2; ++q) {
            const int2 t = reinterpret_cast<const int2 *>(row)[q];
            wt[2 * q + 0] = *reinterpret_cast<const ACC *>(&t.x);
            wt[2 * q + 1] = *reinterpret_cast<const ACC *>(&t.y);
        }
    } else {
#pragma unroll
        for (int q = 0; q < ROWS; ++q) wt[q] = row[q];
    }
}

// packed fp32 pairs (Blackwell FADD2 / FFMA2: two IEEE fp32 operations per issued instruction, same rounding
// as the scalar forms)
__device__ __forceinline__ uint64_t pack2(float lo, float hi)
{
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(uint64_t p, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p)); }
__device__ __forceinline__ uint64_t sub2(uint64_t a, uint64_t b)
{
    uint64_t r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c)
{
    uint64_t r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

// acc[r][v] += x_v * w_r for one frame.  Float: x is pedestal-subtracted exactly, (2^23+x) - (2^23+ped).
template <typename T, typename ACC, int ROWS, int V>
__device__ __forceinline__ void accumulate(const uint32_t (&w)[Pix<T, V>::NW], const ACC (&wt)[ROWS], const float (&pedm)[V],
                                           ACC (&acc)[ROWS][V], uint32_t bsw = 0)
{
    if constexpr (std::is_same<ACC, float>::value && V % 2 == 0) {
#pragma unroll
        for (int v = 0; v < V; v += 2) {
            const uint64_t x = sub2(pack2(Pix<T, V>::getf_biased(w, v, bsw), Pix<T, V>::getf_biased(w, v + 1, bsw)), pack2(pedm[v], pedm[v + 1]));
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                const uint64_t a = fma2(x, pack2(wt[r], wt[r]), pack2(acc[r][v], acc[r][v + 1]));
                unpack2(a, acc[r][v], acc[r][v + 1]);
            }
        }
    } else {
#pragma unroll
        for (int v = 0; v < V; ++v) {
            if constexpr (std::is_same<ACC, float>::value) {
                float x = Pix<T, V>::getf_biased(w, v, bsw) - pedm[v];
#pragma unroll
                for (int r = 0; r < ROWS; ++r) acc[r][v] = fmaf(x, wt[r], acc[r][v]);
            } else {
                int x = (int)Pix<T, V>::geti(w, v, bsw);
#pragma unroll
                for (int r = 0; r < ROWS; ++r) acc[r][v] += x * wt[r];
            }
        }
    }
}

// Integer bins with ONE reference: every frame falls into exactly one phase bin, so its weight row is one-hot
// (+1 or -1 in one row, zeros elsewhere).  The row is the same for every thread (it depends on the frame only):
// branch on it and update that row alone -- V integer multiply-adds per frame instead of ROWS * V.
template <typename T, int ROWS, int V>
__device__ __forceinline__ void accumulate_onehot(const uint32_t (&w)[Pix<T, V>::NW], const int (&wt)[ROWS], int (&acc)[ROWS][V], uint32_t bsw = 0)
{
    int sgn = 0;
#pragma unroll
    for (int r = 0; r < ROWS; ++r) sgn += wt[r];
    int x[V];
#pragma unroll
    for (int v = 0; v < V; ++v) x[v] = (int)Pix<T, V>::geti(w, v, bsw);
    bool done = false;
#pragma unroll
    for (int r = 0; r < ROWS; ++r) {
        if (!done && (wt[r] != 0 || r == ROWS - 1)) {
            done = true;
#pragma unroll
            for (int v = 0; v < V; ++v) acc[r][v] += x[v] * sgn;
        }
    }
}

// window-relative I / Q: turn (I, Q) = (S, C) of reference k back by the angle the absolute-index references are ahead
// (I' = I cos d - Q sin d, Q' = Q cos d + I sin d); rot == nullptr: nothing to do
__device__ __forceinline__ void rotate_iq(const double *rot, int k, double &S, double &C)
{
    if (rot) {
        const double c = rot[2 * k], s = rot[2 * k + 1];
        const double S2 = S * c - C * s;
        C = C * c + S * s;
        S = S2;
    }
}

// ---------------------------------------------------------------------------------------------------
// A4: finalise one pixel from its ROWS sums (already including the pedestal term), all in fp64.
// ---------------------------------------------------------------------------------------------------
template <int ROWS>
__device__ __forceinline__ void finalise_pixel(const FinParams &f, const double (&val)[ROWS], int64_t pixel, int64_t HW)
{
    for (int k = 0; k < f.K; ++k) {
        double S = 0.0, C = 0.0;
        if (f.is_int) {
            const int off = f.row_off[k], end = off + f.n_rows[k];
#pragma unroll
            for (int r = 0; r < ROWS; ++r)
                if (r >= off && r < end) {
                    S += val[r] * f.sw[r];
                    C += val[r] * f.cw[r];
                }
        } else {
#pragma unroll
            for (int r = 0; r + 1 < ROWS; r += 2)
                if (r == 2 * k) {
                    S = val[r];
                    C = val[r + 1];
                }
        }
        rotate_iq(f.rot, k, S, C);
        S *= f.scale;
        C *= f.scale;
        const int64_t o = (int64_t)k * HW + pixel;
        if (f.I) f.I[o] = (float)S;
        if (f.Q) f.Q[o] = (float)C;
        if (f.amp) f.amp[o] = (float)sqrt(S * S + C * C);
        if (f.phase) f.phase[o] = (S == 0.0 && C == 0.0) ? 0.0f : (float)atan2(C, S);
    }
}

// The same with the accumulation kind known at compile time and the sums still in their native type: no
// run-time row tests, no local-memory copy of the sums; K = 1 (the common case) skips the reference loop.
template <int ROWS, bool IS_INT, typename RED>
__device__ __forceinline__ void finalise_pixel_t(const FinParams &f, const RED (&a)[ROWS], double ped, const double (&wsum)[ROWS], int64_t pixel,
                                                 int64_t HW)
{
    auto emit = [&](int k, double S, double C) {
        rotate_iq(f.rot, k, S, C);
        S *= f.scale;
        C *= f.scale;
        const int64_t o = (int64_t)k * HW + pixel;
        if (f.I) f.I[o] = (float)S;
        if (f.Q) f.Q[o] = (float)C;
        if (f.amp) f.amp[o] = (float)sqrt(S * S + C * C);
        if (f.phase) f.phase[o] = (S == 0.0 && C == 0.0) ? 0.0f : (float)atan2(C, S);
    };
    if constexpr (IS_INT) {
        if (f.K == 1) {
            // padding rows carry zero weights and zero sums
            double S = 0.0, C = 0.0;
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                const double v = (double)a[r];
                S = fma(v, f.sw[r], S);
                C = fma(v, f.cw[r], C);
            }
            emit(0, S, C);
        } else {
            for (int k = 0; k < f.K; ++k) {
                const int off = f.row_off[k], end = off + f.n_rows[k];
                double S = 0.0, C = 0.0;
#pragma unroll
                for (int r = 0; r < ROWS; ++r)
                    if (r >= off && r < end) {
                        S = fma((double)a[r], f.sw[r], S);
                        C = fma((double)a[r], f.cw[r], C);
                    }
                emit(k, S, C);
            }
        }
    } else {
#pragma unroll
        for (int k = 0; k < ROWS / 2; ++k)
            if (k < f.K) emit(k, (double)a[2 * k] + ped * wsum[2 * k], (double)a[2 * k + 1] + ped * wsum[2 * k + 1]);
    }
}

// By-value form (the sums travel as a small struct); measured: a real call costs more than the code it saves
// (cfg3 hop 41 -> 46 us), so it stays inline.
template <typename RED, int ROWS>
struct RowVals {
    RED a[ROWS];
};
template <int ROWS, bool IS_INT, typename RED>
__device__ __forceinline__ void finalise_pixel_nl(const FinParams *f, RowVals<RED, ROWS> a, double ped, RowVals<double, ROWS> wsum, int64_t pixel, int64_t HW)
{
    finalise_pixel_t<ROWS, IS_INT, RED>(*f, a.a, ped, wsum.a, pixel, HW);
}

// pixels per thread for a (dtype, rows) pair: at most 16 bytes per load and at most 64 accumulators
constexpr int pick_v(int bytes, int rows)
{
    int v = 16 / bytes;
    while (v * rows > 64 && v > 1) v /= 2;
    return v;
}

}  // namespace qld_dev

// Tensor-core (tcgen05) demodulation path: declarations shared by qld_tc.cu and qld_api.cu.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "qld_internal.h"

struct TcParams {
    int64_t HW;
    int64_t row_bytes;        // H*W*bytes: bytes of one frame
    int32_t N;                // frames in the window
    int32_t bytes;            // 1 (u8) or 2 (u16)
    const int8_t *digits;     // digit tiles, see k_digit_pack
    int64_t *sums_out;        // optional [2K][HW] exact fixed-point sums (Q30 references)
    unsigned int *tile_counter; // device counter for the dynamic tile scheduler: zero on entry
    unsigned int *tile_counter_next; // the next launch's counter, zeroed by this launch (the two alternate)
    int32_t force_T, force_stages, force_kc;   // debug override of the tile shape (qld_debug_set_tile), 0 = automatic
    int32_t big_endian;       // 16-bit samples most significant byte first: the even accumulator row is the high byte
    int32_t bins_rows;        // > 0: integer phase bins (A3'): the B operand holds one signed byte per bin row and frame (16
                              // columns), the epilogue writes the exact int32 rows to bins_out and combines them with fin.sw / fin.cw
    int32_t reserved2;
    int32_t *bins_out;        // [bins_rows padded][HW] int32 (the context's accumulator rows)
    int64_t bins_stride;      // elements between rows of bins_out (HW)
    // unknown-frequency search (qld_dominant_bin): 32 DFT bins per launch (256 columns), running arg-max in spec_amp / spec_bin
    float *spec_amp;          // [HW] largest amplitude so far (read unless spec_first)
    int32_t *spec_bin;        // [HW] its bin
    int32_t spec_q0, spec_nbins, spec_first, reserved3;
    FinParams fin;
};

int qld_tc_columns(int K);                       // N columns of the MMA: 8 per reference, padded to 16
size_t qld_tc_digit_bytes(int K, int N);
// K: references of a fixed-point contraction (8 columns each, padded to 16); K = 2 also describes the 16-column bins contraction
cudaError_t qld_tc_encode_tmap(void *tmaps_out /*2 x 128 B, 64-aligned*/, const void *frames, int64_t row_bytes, int n_frames, int K, int n_sms,
                               const int *force /* {T, stages, kc} or zeros */);
cudaError_t qld_launch_fixed_table_fill(const TableFillParams &p, int32_t *rfix, int n_stride, cudaStream_t st);
// rfix rows (2k, 2k+1) = rint(2^30 * tab[2][n]) from caller-supplied doubles
cudaError_t qld_launch_fixed_from_doubles(const double *tab, int n, int k, int32_t *rfix, int n_stride, cudaStream_t st);
// B operand of the integer-bin contraction from the context's weight table wtab[cap_w][rows] (frames 1..N, entries s mod cap_w)
cudaError_t qld_launch_bins_pack(const int32_t *wtab, int cap_w, int rows, int N, int8_t *digits, cudaStream_t st);
// digit tiles of the DFT bins q_lo .. q_lo + n_bins - 1 of an N-frame window (nu = q/N), 32 bins (256 columns) per pass, steps padded
// to a multiple of 4 (128-frame stages); returns the bytes per pass through *pass_bytes
size_t qld_tc_spectrum_digit_bytes(int N, int n_bins, size_t *pass_bytes);
cudaError_t qld_launch_spectrum_digits(int N, int q_lo, int n_bins, int8_t *digits, cudaStream_t st);
void qld_tc_spectrum_shape(int force_out[3]);     // {T, stages, KC} the search's tensor maps are encoded for
cudaError_t qld_launch_demod_tc_spectrum(const void *tmaps, const TcParams &p, int n_sms, cudaStream_t st);
cudaError_t qld_launch_digit_pack(const int32_t *rfix, int n_stride, int N, int K, int8_t *digits, cudaStream_t st);
cudaError_t qld_launch_demod_tc(const void *tmaps, const TcParams &p, int n_sms, cudaStream_t st);

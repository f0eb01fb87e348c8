// Sliding-window update with every byte moved by the async copy engines (qld_slide.cu): declarations shared with qld_api.cu.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "qld_internal.h"

struct SlideShape {
    int32_t seg;       // contiguous bytes of every frame per tile (0: the kernel does not apply)
    int32_t kc;        // frames per pipeline stage
    int32_t stages;    // frame stages in shared memory
    int32_t nsb;       // per-tile state buffers (stored sums, expired partial sums, pedestal, maps)
};

// rows: padded accumulator rows; n_map_rows: K * (number of maps requested); force: qld_debug_set_tile(which = 2)
// kind: 0 = fp32 (fp64 stored sums, pedestal), 1 = integer bins (int32), 2 = Q1.30 fixed point (int64)
SlideShape qld_slide_shape(int dtype, int kind, int rows, int part, int n_map_rows, int64_t HW, const void *frames, int n_sms, int force);
cudaError_t qld_slide_encode_tmap(void *tmap_out /*128 B, 64-aligned*/, const void *frames, int64_t row_bytes, int cap, const SlideShape &sh);
// p: as for k_demod_stream's sliding launches (runs, acc_out, part / part_sub, ped_in, cum_lo / cum_hi, fin)
cudaError_t qld_launch_slide_bulk(int dtype, int kind, int rows, const void *tmap, const DemodParams &p, const SlideShape &sh,
                                  unsigned int *counter /* zero on entry */, unsigned int *counter_next /* zeroed by the launch */, int n_sms, cudaStream_t st);

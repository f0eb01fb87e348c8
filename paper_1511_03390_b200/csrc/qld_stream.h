// TMA-fed CUDA-core whole-window demodulation (qld_stream.cu): declarations shared with qld_api.cu.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "qld_internal.h"

struct StreamShape {
    int32_t seg;      // contiguous bytes of every frame per tile (0: the streaming kernel does not apply)
    int32_t kc;       // frames per pipeline stage
    int32_t stages;   // shared-memory stages
};

// force_seg / force_kc > 0: debug override of the tile shape (qld_debug_set_tile); it also lifts the frame-size threshold
StreamShape qld_stream_shape(int dtype, int is_int, int rows, int64_t HW, const void *frames, int n_sms, int force_seg = 0, int force_kc = 0);
cudaError_t qld_stream_encode_tmap(void *tmap_out /*128 B, 64-aligned*/, const void *frames, int64_t row_bytes, int cap, const StreamShape &sh);
cudaError_t qld_launch_demod_stream(int dtype, int is_int, int rows, const void *tmap, const DemodParams &p, const StreamShape &sh,
                                    unsigned int *counter /* zero on entry */, unsigned int *counter_next /* zeroed by the launch */, int n_sms, cudaStream_t st);

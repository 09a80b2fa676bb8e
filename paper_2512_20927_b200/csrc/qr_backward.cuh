// qr_backward.cuh -- parameters shared by the qr_backward kernels (qr_backward.cu, qr_backward_tile.cu).
#pragma once
#include "qr_common.cuh"

namespace qr {

struct BackwardParams {
    Cam cam;
    int32_t K, D;
    int64_t N;
    const int32_t* sel_idx;
    const float* sel_w;
    const int32_t* n_sel;
    const float* dL_dmap;
    float* dL_dfeat;
};

// qr_backward_tile.cu: persistent, warp-specialised half-tile kernel (D % 4 == 0).
bool backward_tile_supported(int32_t K, int32_t D);
// qr_backward_mma.cu: the same contraction on tcgen05 (tf32 x 3), D a multiple of 128.
bool backward_mma_supported(int32_t K, int32_t D);
int launch_backward_mma(const BackwardParams& p, cudaStream_t st);
int launch_backward_tile(const BackwardParams& p, cudaStream_t st);

}  // namespace qr

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
    // written by backward_prep_kernel (qr_backward_mma.cu) into the caller's workspace; NULL on the FFMA-only paths
    const int32_t* prep_cnt = nullptr;     // [half tiles][4]: records in pixels 0..63, records, distinct Gaussians,
                                           // 1 = this half tile is left to backward_tile_kernel
    const int32_t* prep_uid = nullptr;     // [half tiles][kBmEntCap] union row -> Gaussian id
    const uint2* prep_ent = nullptr;       // [half tiles][kBmEntCap] {weight bits, union row << 8 | pixel}, pixel order
    const int32_t* prep_nflag = nullptr;   // [1] how many half tiles carry that flag
    bool only_flagged = false;             // backward_tile_kernel: process only half tiles with prep_cnt[..][3] == 1
};

// qr_backward_tile.cu: persistent, warp-specialised half-tile kernel (D % 4 == 0).
bool backward_tile_supported(int32_t K, int32_t D);
// qr_backward_mma.cu: the same contraction on tcgen05 (tf32 x 3), D a multiple of 128.
bool backward_mma_supported(int32_t K, int32_t D);
size_t backward_mma_workspace_bytes(const Cam& cam);
int backward_mma_workspace_view(BackwardParams& p, void* ws, size_t ws_bytes, int* uid_stride, int32_t** seen, int* seen_cells);
int launch_backward_mma(BackwardParams p, void* ws, size_t ws_bytes, cudaStream_t st);
int launch_backward_tile(const BackwardParams& p, cudaStream_t st);

}  // namespace qr

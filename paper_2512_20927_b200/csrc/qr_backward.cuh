// qr_backward.cuh -- parameters shared by the qr_backward kernels (qr_backward.cu, qr_backward_tile.cu).
#pragma once
#include "qr_common.cuh"
#include "qr_sel.cuh"

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
    // tcgen05 path: the selection lists (qr_sel.cuh) -- written by backward_prep_kernel into the caller's workspace, or left
    // there by qr_forward (qr_backward_lists); hdr[5] == 1 marks a half tile left to backward_tile_kernel.  Unset on the
    // FFMA-only paths.
    SelLists sl;
    const int32_t* prep_nflag = nullptr;   // [1] how many half tiles carry that flag
    int32_t* ticket = nullptr;             // tcgen05 contraction: half-tile ticket (zeroed by the launcher)
    bool only_flagged = false;             // backward_tile_kernel: process only half tiles with prep_cnt[..][3] == 1
};

// qr_backward_tile.cu: persistent, warp-specialised half-tile kernel (D % 4 == 0).
bool backward_tile_supported(int32_t K, int32_t D);
// qr_backward_mma.cu: the same contraction on tcgen05 (tf32 x 3), D a multiple of 128.
bool backward_mma_supported(int32_t K, int32_t D);
size_t backward_mma_workspace_bytes(const Cam& cam, int K);
int backward_mma_workspace_view(BackwardParams& p, void* ws, size_t ws_bytes, int32_t** seen, int* seen_cells);
// from_lists: ws is a workspace whose selection lists are already complete (qr_forward's): no numbering pass
int launch_backward_mma(BackwardParams p, void* ws, size_t ws_bytes, cudaStream_t st, bool from_lists);
int launch_backward_tile(const BackwardParams& p, cudaStream_t st);
// backward_prep_kernel alone: numbers each half tile's union of selected Gaussians and writes its entry lists (p.sl) from the
// selection records; *nflag counts the half tiles it left out (more than 5,120 records; their hdr[5] == 1).  qr_topk_forward
// feeds the tcgen05 blend with it.
int launch_backward_prep(const BackwardParams& p, int32_t* nflag, cudaStream_t st);

}  // namespace qr

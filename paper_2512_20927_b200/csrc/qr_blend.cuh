// qr_blend.cuh -- what walk_kernel hands to the blend kernels of qr_forward (qr_forward.cu, qr_blend_mma.cu).
#pragma once
#include "qr_common.cuh"
#include "qr_sel.cuh"

namespace qr {

constexpr int kGroupPx = 8;                  // a pixel group is 4x2 pixels
constexpr int kGroupsPerTile = 32;           // 16x16 tile = 8 row pairs x 4 groups; groups 0..15 = upper 16x8 half
// A record is 12 words (48 B, 16-byte aligned):
//   words 0..7  w^Q of the group's 8 pixels (0 where the pixel did not select the Gaussian; Algorithm 1 line 8)
//   word  8     Gaussian id (-1 in the sentinels that end a list)
//   word  9     bits 0..7: which of the 8 pixels selected it; bits 8..: column of the Gaussian in the union of its
//               16x8 half tile (numbered in order of first selection, any order: the blend sums over them)
//   words 10,11 padding
constexpr int kRecWords = 12;
constexpr int kSentinels = 3;

struct BlendParams {
    Cam cam;
    int32_t K, D, cap, num_tiles;
    int32_t feat_f16 = 0;        // tcgen05 blend: features are fp16 (widened exactly, R14)
    const void* features;
    const int32_t* gcount;       // [tiles * 32] records per group
    const int32_t* ucount;       // [tiles * 2] size of each half tile's union
    const float* rec;            // [tiles * 32][cap][kRecWords]
    const int32_t* n_sel;
    const float* resid;
    float* out_map;
    int32_t* sel_idx;
    float* sel_w;
    int32_t* tile_ticket;
    SelLists sl;                 // tcgen05 blend: the walk's selection lists (qr_sel.cuh); the fields above that describe
                                 // group records are unused there
};

// tcgen05 blend (qr_blend_mma.cu): fp32 features, D a multiple of 256.
bool blend_mma_supported(int32_t D, qr_dtype feat_dtype);
// pdl: launch with programmatic stream serialization behind walk2_kernel (the half tiles' release flags synchronise the
// two); false: a plain launch behind whatever wrote the lists
int launch_blend_mma(const BlendParams& p, cudaStream_t st, bool pdl = true);

}  // namespace qr

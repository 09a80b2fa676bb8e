// qr_preprocess.cu -- EWA projection of 3D Gaussians to screen space (SPEC.md:130-138,
// :163-168; readings R5, R6, R12 of DESIGN.md).  One thread per Gaussian.
//
// Every fp32 operation is spelled with an explicit rounding intrinsic (__fmul_rn, __fadd_rn, __fmaf_rn,
// __fdiv_rn, __fsqrt_rn) in the order DESIGN.md "fp32 decision arithmetic" fixes, so that `depth` (the sort key)
// and the conics that decide list membership do not depend on compiler contraction.
//
// HBM traffic: 44 B in + 48 B out per Gaussian, all through coalesced or 16-byte accesses (AoS rows of 3 floats
// are read as three strided loads; the hardware coalesces a warp's 384 contiguous bytes into 3 full lines).
#include "qr_common.cuh"

namespace qr {

__device__ __forceinline__ float mul(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float sub(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float fdiv(float a, float b) { return __fdiv_rn(a, b); }

// Gaussian i seen by `cam`; results go to slot `o` of the output arrays; the tile rectangle's rows are shifted by `ty_off`
// tiles (0 for a single view; view b of a batch sits b * tiles_y rows down the tall tile grid)
__device__ __forceinline__ void project_one(const Cam& cam, const int64_t i, const int64_t o, const int ty_off,
                                            const float* __restrict__ means, const float* __restrict__ scales,
                                            const float* __restrict__ quats, const float* __restrict__ opac,
                                            float2* __restrict__ mean2d, float4* __restrict__ conic_opac, float* __restrict__ depth,
                                            int4* __restrict__ tile_rect, uint32_t* __restrict__ tiles_touched)
{

    const float mx = means[3 * i], my = means[3 * i + 1], mz = means[3 * i + 2];
    const float* W = cam.w;
    // t = R mu + t_wc: three fma chains, x then y then z (R6: depth must be reproducible)
    float t[3];
#pragma unroll
    for (int r = 0; r < 3; ++r)
        t[r] = __fmaf_rn(W[4 * r + 2], mz, __fmaf_rn(W[4 * r + 1], my, __fmaf_rn(W[4 * r], mx, W[4 * r + 3])));

    const float tz = t[2];
    depth[o] = tz;
    float2 m2 = make_float2(0.f, 0.f);
    float4 co = make_float4(0.f, 0.f, 0.f, 0.f);
    int4 rect = make_int4(0, 0, 0, 0);
    uint32_t touched = 0;

    if (tz > cam.znear) {
        const float4 q = reinterpret_cast<const float4*>(quats)[i];
        const float qw = q.x, qx = q.y, qy = q.z, qz = q.w;
        // R from the unit quaternion (w,x,y,z) -- PAPER.md:79
        float R[9];
        R[0] = sub(1.0f, mul(2.0f, add(mul(qy, qy), mul(qz, qz))));
        R[1] = mul(2.0f, sub(mul(qx, qy), mul(qw, qz)));
        R[2] = mul(2.0f, add(mul(qx, qz), mul(qw, qy)));
        R[3] = mul(2.0f, add(mul(qx, qy), mul(qw, qz)));
        R[4] = sub(1.0f, mul(2.0f, add(mul(qx, qx), mul(qz, qz))));
        R[5] = mul(2.0f, sub(mul(qy, qz), mul(qw, qx)));
        R[6] = mul(2.0f, sub(mul(qx, qz), mul(qw, qy)));
        R[7] = mul(2.0f, add(mul(qy, qz), mul(qw, qx)));
        R[8] = sub(1.0f, mul(2.0f, add(mul(qx, qx), mul(qy, qy))));
        const float s0 = scales[3 * i], s1 = scales[3 * i + 1], s2 = scales[3 * i + 2];
        float M[9];
#pragma unroll
        for (int r = 0; r < 3; ++r) {
            M[3 * r] = mul(R[3 * r], s0); M[3 * r + 1] = mul(R[3 * r + 1], s1); M[3 * r + 2] = mul(R[3 * r + 2], s2);
        }
        float Sig[9];   // Sigma = (R S)(R S)^T
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c)
                Sig[3 * r + c] = add(add(mul(M[3 * r], M[3 * c]), mul(M[3 * r + 1], M[3 * c + 1])),
                                     mul(M[3 * r + 2], M[3 * c + 2]));

        // perspective Jacobian with the clamp of reading R12
        const float limx = fdiv(mul(kJClamp, mul(0.5f, (float)cam.width)), cam.fx);
        const float limy = fdiv(mul(kJClamp, mul(0.5f, (float)cam.height)), cam.fy);
        const float txz = fdiv(t[0], tz), tyz = fdiv(t[1], tz);
        const float cxz = fminf(limx, fmaxf(-limx, txz)), cyz = fminf(limy, fmaxf(-limy, tyz));
        const float tz2 = mul(tz, tz);
        const float J00 = fdiv(cam.fx, tz), J02 = fdiv(-mul(cam.fx, mul(cxz, tz)), tz2);
        const float J11 = fdiv(cam.fy, tz), J12 = fdiv(-mul(cam.fy, mul(cyz, tz)), tz2);
        float Tm[6];   // J * W_rot (2x3)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            Tm[c] = add(mul(J00, W[c]), mul(J02, W[8 + c]));
            Tm[3 + c] = add(mul(J11, W[4 + c]), mul(J12, W[8 + c]));
        }
        float TS[6];   // (J W) Sigma
#pragma unroll
        for (int r = 0; r < 2; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c)
                TS[3 * r + c] = add(add(mul(Tm[3 * r], Sig[c]), mul(Tm[3 * r + 1], Sig[3 + c])),
                                    mul(Tm[3 * r + 2], Sig[6 + c]));
        float cxx = add(add(mul(TS[0], Tm[0]), mul(TS[1], Tm[1])), mul(TS[2], Tm[2]));
        const float cxy = add(add(mul(TS[0], Tm[3]), mul(TS[1], Tm[4])), mul(TS[2], Tm[5]));
        float cyy = add(add(mul(TS[3], Tm[3]), mul(TS[4], Tm[4])), mul(TS[5], Tm[5]));
        cxx = add(cxx, kDilation);   // + 0.3 I
        cyy = add(cyy, kDilation);
        const float det = sub(mul(cxx, cyy), mul(cxy, cxy));
        if (det > 0.0f) {
            co = make_float4(fdiv(cyy, det), fdiv(-cxy, det), fdiv(cxx, det), opac[i]);
            m2 = make_float2(__fmaf_rn(cam.fx, txz, cam.cx), __fmaf_rn(cam.fy, tyz, cam.cy));
            // 3-sigma AABB, inflated by 0.1 % + 0.01 px: the conic that decides membership is an fp32 inverse and its ellipse can
            // reach that far past the AABB of an ill-conditioned cov2d (any superset is correct: rule R4 is per pixel)
            const float ex = add(mul(mul(3.0f, __fsqrt_rn(cxx)), 1.001f), 0.01f), ey = add(mul(mul(3.0f, __fsqrt_rn(cyy)), 1.001f), 0.01f);
            // tile rectangle of the 3-sigma AABB, half-open, clamped to the grid
            const float inv = 1.0f / (float)kTile;   // exact power of two
            const float big = 1.0e6f;
            const float fx0 = floorf(mul(sub(m2.x, ex), inv)), fx1 = floorf(mul(add(m2.x, ex), inv));
            const float fy0 = floorf(mul(sub(m2.y, ey), inv)), fy1 = floorf(mul(add(m2.y, ey), inv));
            const int x0 = min(max((int)fminf(fmaxf(fx0, -big), big), 0), cam.tiles_x);
            const int x1 = min(max((int)fminf(fmaxf(fx1, -big), big) + 1, 0), cam.tiles_x);
            const int y0 = min(max((int)fminf(fmaxf(fy0, -big), big), 0), cam.tiles_y);
            const int y1 = min(max((int)fminf(fmaxf(fy1, -big), big) + 1, 0), cam.tiles_y);
            if (x1 > x0 && y1 > y0) {
                rect = make_int4(x0, y0 + ty_off, x1, y1 + ty_off);
                touched = (uint32_t)((x1 - x0) * (y1 - y0));
            }
        }
    }
    mean2d[o] = m2;
    conic_opac[o] = co;
    tile_rect[o] = rect;
    tiles_touched[o] = touched;
}

__global__ void __launch_bounds__(256)
preprocess_kernel(const Cam cam, const int64_t N, const float* __restrict__ means, const float* __restrict__ scales,
                  const float* __restrict__ quats, const float* __restrict__ opac, float2* __restrict__ mean2d,
                  float4* __restrict__ conic_opac, float* __restrict__ depth, int4* __restrict__ tile_rect,
                  uint32_t* __restrict__ tiles_touched)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    project_one(cam, i, i, 0, means, scales, quats, opac, mean2d, conic_opac, depth, tile_rect, tiles_touched);
}

// B views in one launch (blockIdx.y = view): virtual Gaussian v = b N + i
struct CamBatch { Cam c[QR_MAX_BATCH]; };
__global__ void __launch_bounds__(256)
preprocess_batch_kernel(const __grid_constant__ CamBatch cams, const int64_t N, const float* __restrict__ means,
                        const float* __restrict__ scales, const float* __restrict__ quats, const float* __restrict__ opac,
                        float2* __restrict__ mean2d, float4* __restrict__ conic_opac, float* __restrict__ depth,
                        int4* __restrict__ tile_rect, uint32_t* __restrict__ tiles_touched)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int b = blockIdx.y;
    const Cam& cam = cams.c[b];
    project_one(cam, i, (int64_t)b * N + i, b * cam.tiles_y, means, scales, quats, opac, mean2d, conic_opac, depth, tile_rect,
                tiles_touched);
}

}  // namespace qr

extern "C" int qr_preprocess(const qr_camera* cam, int64_t N, const float* means, const float* scales,
                             const float* quats, const float* opac, float* mean2d, float* conic_opac, float* depth,
                             int32_t* tile_rect, uint32_t* tiles_touched, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (N < 0) return fail(QR_ERR_INVALID_ARG, "N = %lld < 0", (long long)N);
    if (N >= (int64_t(1) << 31)) return fail(QR_ERR_UNSUPPORTED, "N >= 2^31");
    if (N == 0) return QR_OK;
    if (!means || !scales || !quats || !opac || !mean2d || !conic_opac || !depth || !tile_rect || !tiles_touched)
        return fail(QR_ERR_NULL_POINTER, "qr_preprocess: NULL array");
    if (!aligned16(quats) || !aligned16(conic_opac) || !aligned16(tile_rect) || !aligned16(mean2d))
        return fail(QR_ERR_MISALIGNED, "qr_preprocess: quats / mean2d / conic_opac / tile_rect must be 16-byte aligned");
    const Cam k = make_cam(cam);
    const unsigned blocks = (unsigned)((N + 255) / 256);
    preprocess_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(
        k, N, means, scales, quats, opac, reinterpret_cast<float2*>(mean2d), reinterpret_cast<float4*>(conic_opac),
        depth, reinterpret_cast<int4*>(tile_rect), tiles_touched);
    QR_LAUNCH_OK("preprocess_kernel");
    return QR_OK;
}

static int check_batch(const qr_camera* cams, int32_t B)
{
    using namespace qr;
    if (!cams) return fail(QR_ERR_NULL_POINTER, "cameras are NULL");
    if (B < 1 || B > QR_MAX_BATCH) return fail(QR_ERR_INVALID_ARG, "B = %d outside [1, QR_MAX_BATCH]", B);
    for (int b = 0; b < B; ++b) {
        if (int rc = check_cam(cams + b)) return rc;
        if (cams[b].width != cams[0].width || cams[b].height != cams[0].height)
            return fail(QR_ERR_INVALID_ARG, "the views of a batch must have the same image size");
    }
    if (cams[0].height % kTile != 0)
        return fail(QR_ERR_INVALID_ARG, "batched views need height %% 16 == 0 (height = %d)", cams[0].height);
    return QR_OK;
}

extern "C" int qr_batch_camera(const qr_camera* cams, int32_t B, qr_camera* tall)
{
    using namespace qr;
    if (int rc = check_batch(cams, B)) return rc;
    if (!tall) return fail(QR_ERR_NULL_POINTER, "qr_batch_camera: tall is NULL");
    *tall = cams[0];
    tall->height = cams[0].height * B;
    return check_cam(tall);
}

extern "C" int qr_preprocess_batch(const qr_camera* cams, int32_t B, int64_t N, const float* means, const float* scales,
                                   const float* quats, const float* opac, float* mean2d, float* conic_opac, float* depth,
                                   int32_t* tile_rect, uint32_t* tiles_touched, void* stream)
{
    using namespace qr;
    if (int rc = check_batch(cams, B)) return rc;
    if (N < 0) return fail(QR_ERR_INVALID_ARG, "N = %lld < 0", (long long)N);
    if (N * (int64_t)B >= (int64_t(1) << 31)) return fail(QR_ERR_UNSUPPORTED, "B N >= 2^31");
    if (N == 0) return QR_OK;
    if (!means || !scales || !quats || !opac || !mean2d || !conic_opac || !depth || !tile_rect || !tiles_touched)
        return fail(QR_ERR_NULL_POINTER, "qr_preprocess_batch: NULL array");
    if (!aligned16(quats) || !aligned16(conic_opac) || !aligned16(tile_rect) || !aligned16(mean2d))
        return fail(QR_ERR_MISALIGNED, "qr_preprocess_batch: quats / mean2d / conic_opac / tile_rect must be 16-byte aligned");
    CamBatch cb;
    for (int b = 0; b < QR_MAX_BATCH; ++b) cb.c[b] = make_cam(cams + (b < B ? b : 0));
    const dim3 grid((unsigned)((N + 255) / 256), (unsigned)B);
    preprocess_batch_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(
        cb, N, means, scales, quats, opac, reinterpret_cast<float2*>(mean2d), reinterpret_cast<float4*>(conic_opac),
        depth, reinterpret_cast<int4*>(tile_rect), tiles_touched);
    QR_LAUNCH_OK("preprocess_batch_kernel");
    return QR_OK;
}

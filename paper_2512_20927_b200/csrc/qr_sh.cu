// qr_sh_colors: view-dependent RGB of every Gaussian from its spherical-harmonics coefficients -- the RGB payload of
// PAPER.md:940-947 (App. E.6: Q-Render applied to pre-trained 3D-GS models), reading R20.
//
//   colour[i][c] = max(0, 1/2 + sum_k Y_k(dir_i) sh[i][k][c]),  dir_i = (mean_i - centre) / |mean_i - centre|,
//   centre = -R^T t,  Y_k = the real harmonics of degree <= 3, ordered (l, m = -l..l), Condon-Shortley phase kept.
//
// HBM-bound: 12 + 12 (degree + 1)^2 + 12 bytes per Gaussian (216 at degree 3).  A CTA owns 128 consecutive Gaussians:
// their coefficient rows are one contiguous block, copied with coalesced 16-byte loads into shared memory (row stride
// padded to an odd number of words: thread = Gaussian then reads its row without bank conflicts), and the colours leave
// through shared memory the same way.
#include "qr_common.cuh"

namespace qr {

constexpr int kShThreads = 128;

// constants of R20 (closed forms in the comments; fp32 literals rounded from them)
constexpr float kY0 = 0.28209479177387814f;     // 1 / (2 sqrt(pi))
constexpr float kY1 = 0.4886025119029199f;      // sqrt(3 / (4 pi))
constexpr float kY2a = 1.0925484305920792f;     // sqrt(15 / pi) / 2
constexpr float kY2b = 0.31539156525252005f;    // sqrt(5 / pi) / 4
constexpr float kY2c = 0.5462742152960396f;     // sqrt(15 / pi) / 4
constexpr float kY3a = 0.5900435899266435f;     // sqrt(35 / (2 pi)) / 4
constexpr float kY3b = 2.890611442640554f;      // sqrt(105 / pi) / 2
constexpr float kY3c = 0.4570457994644658f;     // sqrt(21 / (2 pi)) / 4
constexpr float kY3d = 0.3731763325901154f;     // sqrt(7 / pi) / 4
constexpr float kY3e = 1.445305721320277f;      // sqrt(105 / pi) / 4

template <int DEG>
__global__ void __launch_bounds__(kShThreads)
sh_colors_kernel(const float cx, const float cy, const float cz, const int64_t N, const float* __restrict__ means,
                 const float* __restrict__ sh, float* __restrict__ colors)
{
    constexpr int NB = (DEG + 1) * (DEG + 1), ROW = NB * 3, PITCH = ROW | 1;      // odd pitch: conflict-free rows
    __shared__ float s_sh[kShThreads * PITCH];
    __shared__ float s_io[kShThreads * 3];
    const int t = threadIdx.x;
    const int64_t g0 = (int64_t)blockIdx.x * kShThreads;
    const int n = (int)min((int64_t)kShThreads, N - g0);
    // the block's coefficients: n * ROW consecutive floats (16-byte loads where the block start is aligned)
    const float* src = sh + g0 * ROW;
    const int total = n * ROW;
    if ((reinterpret_cast<uintptr_t>(src) & 15) == 0) {
        // every load of the thread is issued before the first shared-memory store
        constexpr int V = (ROW * kShThreads / 4 + kShThreads - 1) / kShThreads;
        float4 v[V];
#pragma unroll
        for (int i = 0; i < V; ++i) {
            const int k = (t + i * kShThreads) * 4;
            v[i] = k + 4 <= total ? __ldg(reinterpret_cast<const float4*>(src + k)) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int i = 0; i < V; ++i) {
            const int k = (t + i * kShThreads) * 4;
            if (k + 4 <= total) {
                const float e[4] = { v[i].x, v[i].y, v[i].z, v[i].w };
#pragma unroll
                for (int u = 0; u < 4; ++u) s_sh[((k + u) / ROW) * PITCH + (k + u) % ROW] = e[u];
            } else {
                for (int u = k; u < total; ++u) s_sh[(u / ROW) * PITCH + u % ROW] = __ldg(src + u);
            }
        }
    } else {
        for (int k = t; k < total; k += kShThreads) s_sh[(k / ROW) * PITCH + k % ROW] = __ldg(src + k);
    }
    for (int k = t; k < n * 3; k += kShThreads) s_io[k] = __ldg(means + g0 * 3 + k);
    __syncthreads();
    float r = 0.f, g = 0.f, b = 0.f;
    if (t < n) {
        float x = s_io[3 * t] - cx, y = s_io[3 * t + 1] - cy, z = s_io[3 * t + 2] - cz;
        const float n2 = x * x + y * y + z * z;
        const float* c = s_sh + t * PITCH;
        r = 0.5f + kY0 * c[0]; g = 0.5f + kY0 * c[1]; b = 0.5f + kY0 * c[2];
        if (DEG >= 1 && n2 > 0.f) {           // a Gaussian at the camera centre keeps the constant term only
            const float inv = 1.0f / sqrtf(n2);
            x *= inv; y *= inv; z *= inv;
            float Y[16];
            Y[1] = -kY1 * y; Y[2] = kY1 * z; Y[3] = -kY1 * x;
            if (DEG >= 2) {
                const float xx = x * x, yy = y * y, zz = z * z;
                Y[4] = kY2a * x * y; Y[5] = -kY2a * y * z; Y[6] = kY2b * (2.f * zz - xx - yy);
                Y[7] = -kY2a * x * z; Y[8] = kY2c * (xx - yy);
                if (DEG >= 3) {
                    Y[9] = -kY3a * y * (3.f * xx - yy); Y[10] = kY3b * x * y * z;
                    Y[11] = -kY3c * y * (4.f * zz - xx - yy); Y[12] = kY3d * z * (2.f * zz - 3.f * xx - 3.f * yy);
                    Y[13] = -kY3c * x * (4.f * zz - xx - yy); Y[14] = kY3e * z * (xx - yy);
                    Y[15] = -kY3a * x * (xx - 3.f * yy);
                }
            }
#pragma unroll
            for (int k = 1; k < NB; ++k) { r += Y[k] * c[3 * k]; g += Y[k] * c[3 * k + 1]; b += Y[k] * c[3 * k + 2]; }
        }
        r = fmaxf(r, 0.f); g = fmaxf(g, 0.f); b = fmaxf(b, 0.f);
    }
    __syncthreads();
    if (t < n) { s_io[3 * t] = r; s_io[3 * t + 1] = g; s_io[3 * t + 2] = b; }
    __syncthreads();
    for (int k = t; k < n * 3; k += kShThreads) colors[g0 * 3 + k] = s_io[k];
}

}  // namespace qr

extern "C" int qr_sh_colors(const qr_camera* cam, int64_t N, int32_t degree, const float* means, const float* sh,
                            float* colors, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (N < 0) return fail(QR_ERR_INVALID_ARG, "qr_sh_colors: N = %lld < 0", (long long)N);
    if (degree < 0 || degree > 3) return fail(QR_ERR_INVALID_ARG, "qr_sh_colors: degree = %d outside [0, 3]", degree);
    if (N == 0) return QR_OK;
    if (!means || !sh || !colors) return fail(QR_ERR_NULL_POINTER, "qr_sh_colors: NULL array");
    // camera centre = -R^T t, in fp64 on the host
    const float* w = cam->world_to_cam;
    float c[3];
    for (int j = 0; j < 3; ++j)
        c[j] = (float)-((double)w[0 + j] * (double)w[3] + (double)w[4 + j] * (double)w[7] + (double)w[8 + j] * (double)w[11]);
    const unsigned blocks = (unsigned)((N + kShThreads - 1) / kShThreads);
    cudaStream_t st = (cudaStream_t)stream;
    switch (degree) {
    case 0: sh_colors_kernel<0><<<blocks, kShThreads, 0, st>>>(c[0], c[1], c[2], N, means, sh, colors); break;
    case 1: sh_colors_kernel<1><<<blocks, kShThreads, 0, st>>>(c[0], c[1], c[2], N, means, sh, colors); break;
    case 2: sh_colors_kernel<2><<<blocks, kShThreads, 0, st>>>(c[0], c[1], c[2], N, means, sh, colors); break;
    default: sh_colors_kernel<3><<<blocks, kShThreads, 0, st>>>(c[0], c[1], c[2], N, means, sh, colors); break;
    }
    QR_LAUNCH_OK("sh_colors_kernel");
    return QR_OK;
}

// qr_neighbours.cu -- the two steps either side of the render path:
//
//   qr_devoxelize / qr_devoxelize_backward   PAPER.md:1121-1179 (Listing 3): per-unique-voxel predictions -> per-Gaussian
//       features F (what qr_forward reads), and the adjoint that carries dL/dF (what qr_backward writes) back to the
//       unique voxels.  Step 1 of the listing (expansion by the inverse index) is never materialised: a warp owns one
//       Gaussian, walks its voxels and reads each voxel's row straight from the unique table (row = C contiguous floats,
//       one coalesced burst), reducing in registers (mean or componentwise max).  HBM-bound gather + segmented reduce.
//   qr_mask_loss                             PAPER.md:216-228 (Eq. 2), reading R19: mean pooling of the rendered
//       map over each mask, cosine-similarity InfoNCE against the S target embeddings, and dL/dmap -- three small kernels
//       around one read of the map and one write of dL/dmap.
#include "qr_common.cuh"

namespace qr {

constexpr int kNbMaxC = QR_MAX_D;          // channels a lane's registers cover: 16 x 32

// ---------------------------------------------------------------------------------------------------------------
// de-voxelisation: warp = Gaussian, lane = channels lane, lane + 32, ...
// off = INCLUSIVE prefix sum of the counts (Gaussian g owns voxels [off[g-1], off[g]), off[-1] = 0)
// ---------------------------------------------------------------------------------------------------------------
template <bool MAX>
__global__ void __launch_bounds__(256) devoxelize_kernel(const int64_t G, const int C, const float* __restrict__ uni,
                                                         const int64_t* __restrict__ inv, const uint64_t* __restrict__ off,
                                                         float* __restrict__ gs, int32_t* __restrict__ argmax)
{
    const int lane = threadIdx.x & 31;
    const int64_t g = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (g >= G) return;
    const int64_t v0 = g > 0 ? (int64_t)off[g - 1] : 0, v1 = (int64_t)off[g];
    float acc[kNbMaxC / 32];
    int32_t am[kNbMaxC / 32];
#pragma unroll
    for (int j = 0; j < kNbMaxC / 32; ++j) { acc[j] = 0.0f; am[j] = -1; }
    for (int64_t v = v0; v < v1; ++v) {
        const float* row = uni + inv[v] * C;
#pragma unroll
        for (int j = 0; j < kNbMaxC / 32; ++j) {
            const int c = j * 32 + lane;
            if (c < C) {
                const float x = __ldg(row + c);
                if (MAX) { if (am[j] < 0 || x > acc[j]) { acc[j] = x; am[j] = (int32_t)v; } }     // first voxel wins a tie
                else acc[j] = __fadd_rn(acc[j], x);
            }
        }
    }
    const float n = (float)(v1 - v0);
#pragma unroll
    for (int j = 0; j < kNbMaxC / 32; ++j) {
        const int c = j * 32 + lane;
        if (c < C) {
            gs[g * C + c] = (MAX || v1 == v0) ? acc[j] : __fdiv_rn(acc[j], n);
            if (MAX) argmax[g * C + c] = am[j];
        }
    }
}

// the same for C % 4 == 0: lane = 4 consecutive channels of every 128-channel slab (one 512-byte row segment per warp
// instruction), two voxels in flight
template <bool MAX>
__global__ void __launch_bounds__(256) devoxelize_vec_kernel(const int64_t G, const int C, const float* __restrict__ uni,
                                                             const int64_t* __restrict__ inv, const uint64_t* __restrict__ off,
                                                             float* __restrict__ gs, int32_t* __restrict__ argmax)
{
    constexpr int NS = kNbMaxC / 128;
    const int lane = threadIdx.x & 31;
    const int64_t g = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (g >= G) return;
    const int64_t v0 = g > 0 ? (int64_t)off[g - 1] : 0, v1 = (int64_t)off[g];
    float acc[NS][4];
    int32_t am[NS][4];
#pragma unroll
    for (int j = 0; j < NS; ++j)
#pragma unroll
        for (int q = 0; q < 4; ++q) { acc[j][q] = 0.0f; am[j][q] = -1; }
    auto load = [&](int64_t v, float4 (&x)[NS]) {
        const float4* row = reinterpret_cast<const float4*>(uni + inv[v] * C);
#pragma unroll
        for (int j = 0; j < NS; ++j)
            if ((j * 32 + lane) * 4 < C) x[j] = __ldg(row + j * 32 + lane);
    };
    auto apply = [&](int64_t v, const float4 (&x)[NS]) {
#pragma unroll
        for (int j = 0; j < NS; ++j) {
            if ((j * 32 + lane) * 4 < C) {
                const float xs[4] = { x[j].x, x[j].y, x[j].z, x[j].w };
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    if (MAX) { if (am[j][q] < 0 || xs[q] > acc[j][q]) { acc[j][q] = xs[q]; am[j][q] = (int32_t)v; } }
                    else acc[j][q] = __fadd_rn(acc[j][q], xs[q]);
                }
            }
        }
    };
    int64_t v = v0;
    for (; v + 1 < v1; v += 2) {
        float4 xa[NS], xb[NS];
        load(v, xa); load(v + 1, xb);
        apply(v, xa); apply(v + 1, xb);
    }
    if (v < v1) { float4 xa[NS]; load(v, xa); apply(v, xa); }
    const float n = (float)(v1 - v0);
#pragma unroll
    for (int j = 0; j < NS; ++j) {
        const int c = (j * 32 + lane) * 4;
        if (c < C) {
            float o[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) o[q] = (MAX || v1 == v0) ? acc[j][q] : __fdiv_rn(acc[j][q], n);
            *reinterpret_cast<float4*>(gs + g * C + c) = make_float4(o[0], o[1], o[2], o[3]);
            if (MAX) *reinterpret_cast<int4*>(argmax + g * C + c) = make_int4(am[j][0], am[j][1], am[j][2], am[j][3]);
        }
    }
}

template <bool MAX>
__global__ void __launch_bounds__(256) devoxelize_backward_kernel(const int64_t G, const int C, const int64_t* __restrict__ inv,
                                                                  const uint64_t* __restrict__ off, const int32_t* __restrict__ argmax,
                                                                  const float* __restrict__ d_gs, float* __restrict__ d_uni)
{
    const int lane = threadIdx.x & 31;
    const int64_t g = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (g >= G) return;
    const int64_t v0 = g > 0 ? (int64_t)off[g - 1] : 0, v1 = (int64_t)off[g];
    if (v1 == v0) return;
    if (MAX) {
        for (int c = lane; c < C; c += 32) {
            const int32_t v = argmax[g * C + c];
            if (v >= 0) atomicAdd(d_uni + inv[v] * C + c, d_gs[g * C + c]);
        }
        return;
    }
    const float n = (float)(v1 - v0);
    float d[kNbMaxC / 32];
#pragma unroll
    for (int j = 0; j < kNbMaxC / 32; ++j) {
        const int c = j * 32 + lane;
        d[j] = c < C ? __fdiv_rn(d_gs[g * C + c], n) : 0.0f;
    }
    for (int64_t v = v0; v < v1; ++v) {
        float* row = d_uni + inv[v] * C;
#pragma unroll
        for (int j = 0; j < kNbMaxC / 32; ++j) {
            const int c = j * 32 + lane;
            if (c < C) atomicAdd(row + c, d[j]);          // one coalesced reduction per (voxel, 32 channels)
        }
    }
}

static int check_devox(int64_t U, int32_t C, int64_t G, int32_t reduce, const char* who)
{
    if (U < 0 || G < 0) return fail(QR_ERR_INVALID_ARG, "%s: negative size", who);
    if (C < 1) return fail(QR_ERR_INVALID_ARG, "%s: C = %d < 1", who, C);
    if (C > kNbMaxC) return fail(QR_ERR_UNSUPPORTED, "%s: C = %d > %d", who, C, kNbMaxC);
    if (reduce != QR_REDUCE_MEAN && reduce != QR_REDUCE_MAX) return fail(QR_ERR_INVALID_ARG, "%s: reduce must be QR_REDUCE_MEAN or QR_REDUCE_MAX", who);
    return QR_OK;
}

}  // namespace qr

extern "C" size_t qr_devoxelize_workspace_bytes(int64_t G)
{
    if (G < 0) return 0;
    return qr::align_up((size_t)(G > 0 ? G : 1) * 8, 256) + qr::align_up((size_t)qr::scan_blocks(G) * 8, 256);
}

extern "C" int qr_devoxelize(int64_t U, int32_t C, int64_t G, const float* uni_pred, const int64_t* inverse_indices,
                             const uint32_t* num_voxels_per_g, int32_t reduce, float* gs_pred, int32_t* argmax, void* ws,
                             size_t ws_bytes, void* stream)
{
    using namespace qr;
    if (int rc = check_devox(U, C, G, reduce, "qr_devoxelize")) return rc;
    if (G == 0) return QR_OK;
    if (!uni_pred || !inverse_indices || !num_voxels_per_g || !gs_pred || !ws) return fail(QR_ERR_NULL_POINTER, "qr_devoxelize: NULL argument");
    if (reduce == QR_REDUCE_MAX && !argmax) return fail(QR_ERR_NULL_POINTER, "qr_devoxelize: argmax is NULL (needed for reduce = max)");
    if (ws_bytes < qr_devoxelize_workspace_bytes(G)) return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_devoxelize: workspace too small");
    cudaStream_t st = (cudaStream_t)stream;
    uint64_t* off = static_cast<uint64_t*>(ws);
    uint64_t* sums = reinterpret_cast<uint64_t*>(static_cast<char*>(ws) + align_up((size_t)G * 8, 256));
    if (int rc = launch_inclusive_scan_u32(num_voxels_per_g, G, off, sums, st)) return rc;      // Listing 3: offset = cumsum(counts)
    const unsigned blocks = (unsigned)((G + 7) / 8);
    const bool vec = C % 4 == 0 && aligned16(uni_pred) && aligned16(gs_pred) && (reduce != QR_REDUCE_MAX || aligned16(argmax));
    if (vec) {
        if (reduce == QR_REDUCE_MAX) devoxelize_vec_kernel<true><<<blocks, 256, 0, st>>>(G, C, uni_pred, inverse_indices, off, gs_pred, argmax);
        else devoxelize_vec_kernel<false><<<blocks, 256, 0, st>>>(G, C, uni_pred, inverse_indices, off, gs_pred, argmax);
    } else if (reduce == QR_REDUCE_MAX) devoxelize_kernel<true><<<blocks, 256, 0, st>>>(G, C, uni_pred, inverse_indices, off, gs_pred, argmax);
    else devoxelize_kernel<false><<<blocks, 256, 0, st>>>(G, C, uni_pred, inverse_indices, off, gs_pred, argmax);
    QR_LAUNCH_OK("devoxelize_kernel");
    return QR_OK;
}

extern "C" int qr_devoxelize_backward(int64_t U, int32_t C, int64_t G, const int64_t* inverse_indices, int32_t reduce,
                                      const int32_t* argmax, const float* d_gs, float* d_uni, const void* ws, size_t ws_bytes,
                                      void* stream)
{
    using namespace qr;
    if (int rc = check_devox(U, C, G, reduce, "qr_devoxelize_backward")) return rc;
    if (G == 0) return QR_OK;
    if (!inverse_indices || !d_gs || !d_uni || !ws) return fail(QR_ERR_NULL_POINTER, "qr_devoxelize_backward: NULL argument");
    if (reduce == QR_REDUCE_MAX && !argmax) return fail(QR_ERR_NULL_POINTER, "qr_devoxelize_backward: argmax is NULL");
    if (ws_bytes < qr_devoxelize_workspace_bytes(G)) return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_devoxelize_backward: workspace too small");
    cudaStream_t st = (cudaStream_t)stream;
    const uint64_t* off = static_cast<const uint64_t*>(ws);          // the offsets qr_devoxelize left there
    const unsigned blocks = (unsigned)((G + 7) / 8);
    if (reduce == QR_REDUCE_MAX) devoxelize_backward_kernel<true><<<blocks, 256, 0, st>>>(G, C, inverse_indices, off, argmax, d_gs, d_uni);
    else devoxelize_backward_kernel<false><<<blocks, 256, 0, st>>>(G, C, inverse_indices, off, argmax, d_gs, d_uni);
    QR_LAUNCH_OK("devoxelize_backward_kernel");
    return QR_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// mask-pooled contrastive loss (Eq. 2; reading R19)
// workspace: sum[S][D] fp32 (pooled sums, then the per-mask gradient rows g), cnt[S] int32, valid[S] int32, norm[S] fp32
// ---------------------------------------------------------------------------------------------------------------
namespace qr {

struct MaskWs { float* sum; int32_t* cnt; int32_t* valid; float* norm; size_t total; };
static MaskWs mask_ws(void* ws, int S, int D)
{
    MaskWs w;
    char* b = static_cast<char*>(ws);
    size_t o = 0;
    w.sum = reinterpret_cast<float*>(b + o);     o = align_up(o + (size_t)S * D * 4, 256);
    w.cnt = reinterpret_cast<int32_t*>(b + o);   o = align_up(o + (size_t)S * 4, 256);
    w.valid = reinterpret_cast<int32_t*>(b + o); o = align_up(o + (size_t)S * 4, 256);
    w.norm = reinterpret_cast<float*>(b + o);    o = align_up(o + (size_t)S * 4, 256);
    w.total = o;
    return w;
}

// warp = a strip of 64 consecutive pixels (raster order); lane = channels lane, lane + 32, ...  Masks are spatially coherent, so
// the warp accumulates a run of equal mask ids in registers and flushes it with one coalesced reduction per 32 channels.
constexpr int kPoolStrip = 64;
__global__ void __launch_bounds__(256) mask_pool_kernel(const int64_t P, const int D, const int S, const float* __restrict__ map,
                                                        const int32_t* __restrict__ mask_id, float* __restrict__ sum, int32_t* __restrict__ cnt)
{
    const int lane = threadIdx.x & 31;
    const int64_t strip = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int64_t p0 = strip * kPoolStrip, p1 = min(P, p0 + kPoolStrip);
    if (p0 >= P) return;
    constexpr int NS = kNbMaxC / 128;          // lane = 4 consecutive channels of every 128-channel slab (D % 4 == 0)
    float4 acc[NS];
#pragma unroll
    for (int j = 0; j < NS; ++j) acc[j] = make_float4(0.f, 0.f, 0.f, 0.f);
    int cur = -1, run = 0;
    auto flush = [&]() {
        if (cur >= 0 && cur < S && run > 0) {
#pragma unroll
            for (int j = 0; j < NS; ++j) {
                const int c = (j * 32 + lane) * 4;
                if (c < D) {
                    float* dst = sum + (int64_t)cur * D + c;
                    atomicAdd(dst, acc[j].x); atomicAdd(dst + 1, acc[j].y); atomicAdd(dst + 2, acc[j].z); atomicAdd(dst + 3, acc[j].w);
                }
            }
            if (lane == 0) atomicAdd(cnt + cur, run);
        }
#pragma unroll
        for (int j = 0; j < NS; ++j) acc[j] = make_float4(0.f, 0.f, 0.f, 0.f);
        run = 0;
    };
    for (int64_t p = p0; p < p1; ++p) {
        const int s = mask_id[p];
        if (s != cur) { flush(); cur = s; }
        if (s >= 0 && s < S) {
            ++run;
            const float4* row = reinterpret_cast<const float4*>(map + p * D);
#pragma unroll
            for (int j = 0; j < NS; ++j) {
                if ((j * 32 + lane) * 4 < D) {
                    const float4 x = __ldg(row + j * 32 + lane);
                    acc[j].x += x.x; acc[j].y += x.y; acc[j].z += x.z; acc[j].w += x.w;
                }
            }
        }
    }
    flush();
}

// one CTA per mask: pooled = sum / count (in place), its norm, validity
__global__ void __launch_bounds__(256) mask_mean_kernel(const int D, float* __restrict__ sum, const int32_t* __restrict__ cnt,
                                                        int32_t* __restrict__ valid, float* __restrict__ norm)
{
    __shared__ float red[8];
    const int s = blockIdx.x, n = cnt[s];
    float n2 = 0.0f;
    for (int d = threadIdx.x; d < D; d += 256) {
        const float v = n > 0 ? sum[(int64_t)s * D + d] / (float)n : 0.0f;
        sum[(int64_t)s * D + d] = v;
        n2 += v * v;
    }
    for (int o = 16; o > 0; o >>= 1) n2 += __shfl_xor_sync(0xffffffffu, n2, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = n2;
    __syncthreads();
    if (threadIdx.x == 0) {
        float t = 0.0f;
        for (int w = 0; w < 8; ++w) t += red[w];
        norm[s] = sqrtf(t);
        valid[s] = (n > 0 && t > 0.0f) ? 1 : 0;
    }
}

// one CTA per mask: cosine similarities to all S targets, log-sum-exp loss, gradient row g_s (written over pooled_s AFTER the
// whole grid has read the pooled rows it needs: a CTA only reads its OWN pooled row, so in place is safe)
__global__ void __launch_bounds__(256) mask_grad_kernel(const int D, const int S, const float* __restrict__ targets, float* __restrict__ pooled,
                                                        const int32_t* __restrict__ cnt, const int32_t* __restrict__ valid,
                                                        const float* __restrict__ norm, float* __restrict__ loss, float* __restrict__ loss_s)
{
    extern __shared__ float sm[];           // p[D], c[S], tn[S], coef[S]
    float* p = sm; float* c = p + D; float* tn = c + S; float* coef = tn + S;
    __shared__ float red[8];
    __shared__ float s_mx, s_Z;
    __shared__ int s_eff;
    const int s = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int eff = 0;
    for (int j = tid; j < S; j += 256) eff += valid[j];
    for (int o = 16; o > 0; o >>= 1) eff += __shfl_xor_sync(0xffffffffu, eff, o);
    if (lane == 0) red[warp] = (float)eff;
    for (int d = tid; d < D; d += 256) p[d] = pooled[(int64_t)s * D + d];
    __syncthreads();
    if (tid == 0) { int t = 0; for (int w = 0; w < 8; ++w) t += (int)red[w]; s_eff = t; }
    __syncthreads();
    if (!valid[s]) {
        for (int d = tid; d < D; d += 256) pooled[(int64_t)s * D + d] = 0.0f;       // no loss, no gradient
        if (tid == 0) loss_s[s] = 0.0f;
        return;
    }
    const float np = norm[s];
    for (int j = warp; j < S; j += 8) {                       // warp per target: dot and norm
        float dot = 0.0f, n2 = 0.0f;
        for (int d = lane; d < D; d += 32) { const float t = __ldg(targets + (int64_t)j * D + d); dot += p[d] * t; n2 += t * t; }
        for (int o = 16; o > 0; o >>= 1) { dot += __shfl_xor_sync(0xffffffffu, dot, o); n2 += __shfl_xor_sync(0xffffffffu, n2, o); }
        if (lane == 0) { tn[j] = sqrtf(n2); c[j] = dot / (np * sqrtf(n2)); }
    }
    __syncthreads();
    if (tid == 0) {                                           // S is small (masks per frame): a serial soft-max is negligible
        float mx = -3.0e38f;
        for (int j = 0; j < S; ++j) mx = fmaxf(mx, c[j]);
        float Z = 0.0f;
        for (int j = 0; j < S; ++j) Z += expf(c[j] - mx);
        s_mx = mx; s_Z = Z;
        const float l = (mx + logf(Z)) - c[s];
        loss_s[s] = l;
        atomicAdd(loss, l / (float)s_eff);
    }
    __syncthreads();
    for (int j = tid; j < S; j += 256) coef[j] = expf(c[j] - s_mx) / s_Z - (j == s ? 1.0f : 0.0f);
    __syncthreads();
    const float scale = 1.0f / ((float)cnt[s] * (float)s_eff);
    for (int d = tid; d < D; d += 256) {
        float g = 0.0f;
        for (int j = 0; j < S; ++j) g += coef[j] * (__ldg(targets + (int64_t)j * D + d) / tn[j] - c[j] * p[d] / np);
        pooled[(int64_t)s * D + d] = g / np * scale;          // d L / d map of every pixel of this mask
    }
}

// d_map[p,:] = g[mask_id[p],:] (0 outside every mask): one float4 per thread, streaming stores
__global__ void __launch_bounds__(256) mask_dmap_kernel(const int64_t P, const int D, const int S, const int32_t* __restrict__ mask_id,
                                                        const float* __restrict__ g, float* __restrict__ d_map)
{
    const int D4 = D >> 2;
    const int64_t n4 = P * D4, stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
        const int64_t p = i / D4;
        const int c4 = (int)(i - p * D4);
        const int s = mask_id[p];
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        if (s >= 0 && s < S) v = __ldg(reinterpret_cast<const float4*>(g + (int64_t)s * D) + c4);
        __stcs(reinterpret_cast<float4*>(d_map) + i, v);
    }
}

}  // namespace qr

extern "C" size_t qr_mask_loss_workspace_bytes(int32_t S, int32_t D)
{
    if (S < 1 || D < 1) return 0;
    return qr::mask_ws(nullptr, S, D).total;
}

extern "C" int qr_mask_loss(const qr_camera* cam, int32_t D, int32_t S, const float* map, const int32_t* mask_id,
                            const float* targets, float* loss, float* loss_per_mask, float* d_map, void* ws, size_t ws_bytes,
                            void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (D < 4 || D % 4 != 0) return fail(QR_ERR_UNSUPPORTED, "qr_mask_loss: D = %d must be a positive multiple of 4", D);
    if (D > kNbMaxC) return fail(QR_ERR_UNSUPPORTED, "qr_mask_loss: D = %d > %d", D, kNbMaxC);
    if (S < 1 || S > QR_MAX_MASKS) return fail(QR_ERR_INVALID_ARG, "qr_mask_loss: S = %d outside [1, QR_MAX_MASKS]", S);
    if (!map || !mask_id || !targets || !loss || !loss_per_mask || !d_map || !ws) return fail(QR_ERR_NULL_POINTER, "qr_mask_loss: NULL argument");
    if (!aligned16(map) || !aligned16(d_map) || !aligned16(ws)) return fail(QR_ERR_MISALIGNED, "qr_mask_loss: map / d_map / ws must be 16-byte aligned");
    const MaskWs w = mask_ws(ws, S, D);
    if (ws_bytes < w.total) return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_mask_loss: workspace %zu < %zu bytes", ws_bytes, w.total);
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t P = (int64_t)cam->width * cam->height;
    QR_CUDA_OK(cudaMemsetAsync(ws, 0, w.total, st));
    QR_CUDA_OK(cudaMemsetAsync(loss, 0, sizeof(float), st));
    const int64_t strips = (P + kPoolStrip - 1) / kPoolStrip;
    mask_pool_kernel<<<(unsigned)((strips + 7) / 8), 256, 0, st>>>(P, D, S, map, mask_id, w.sum, w.cnt);
    QR_LAUNCH_OK("mask_pool_kernel");
    mask_mean_kernel<<<(unsigned)S, 256, 0, st>>>(D, w.sum, w.cnt, w.valid, w.norm);
    QR_LAUNCH_OK("mask_mean_kernel");
    const size_t smem = ((size_t)D + 3 * (size_t)S) * 4;
    mask_grad_kernel<<<(unsigned)S, 256, smem, st>>>(D, S, targets, w.sum, w.cnt, w.valid, w.norm, loss, loss_per_mask);
    QR_LAUNCH_OK("mask_grad_kernel");
    mask_dmap_kernel<<<(unsigned)(sm_count() * 8), 256, 0, st>>>(P, D, S, mask_id, w.sum, d_map);
    QR_LAUNCH_OK("mask_dmap_kernel");
    return QR_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// qr_mask_loss_static: qr_mask_loss for callers that cannot allocate (code under CUDA graph capture, serving loops,
// harnesses that forbid cudaMalloc).  The same four kernels, with the workspace (per-mask sums, counts, flags, norms) in a
// file-scope device array of QR_STATIC_SCRATCH_BYTES instead of a caller-provided buffer; every GPU that loads the library
// holds the array until exit.  In HOST code the array's name is a host-side stand-in, not a device address: the address the
// kernels get comes from cudaGetSymbolAddress, asked for once per device with that device current.
// ---------------------------------------------------------------------------------------------------------------
#include <mutex>

static __device__ __align__(256) unsigned char g_mask_scratch[QR_STATIC_SCRATCH_BYTES];

namespace qr {

constexpr int kStaticMaxDevices = 64;

// device address of g_mask_scratch on the CURRENT device (nullptr + error state on failure)
static int static_scratch_ptr(void** out)
{
    static std::mutex mu;
    static void* ptr[kStaticMaxDevices] = {};
    int dev = -1;
    QR_CUDA_OK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(QR_ERR_UNSUPPORTED, "qr_mask_loss_static: device ordinal %d >= %d", dev, kStaticMaxDevices);
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_mask_scratch);
        if (e != cudaSuccess || !p)
            return fail(QR_ERR_CUDA, "qr_mask_loss_static: cudaGetSymbolAddress failed on device %d: %s", dev, cudaGetErrorString(e));
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return QR_OK;
}

}  // namespace qr

extern "C" int qr_mask_loss_static(const qr_camera* cam, int32_t D, int32_t S, const float* map, const int32_t* mask_id,
                                   const float* targets, float* loss, float* loss_per_mask, float* d_map, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (D < 4 || D % 4 != 0) return fail(QR_ERR_UNSUPPORTED, "qr_mask_loss_static: D = %d must be a positive multiple of 4", D);
    if (D > kNbMaxC) return fail(QR_ERR_UNSUPPORTED, "qr_mask_loss_static: D = %d > %d", D, kNbMaxC);
    if (S < 1 || S > QR_MAX_MASKS) return fail(QR_ERR_INVALID_ARG, "qr_mask_loss_static: S = %d outside [1, QR_MAX_MASKS]", S);
    const size_t need = mask_ws(nullptr, S, D).total;
    if (need > (size_t)QR_STATIC_SCRATCH_BYTES)
        return fail(QR_ERR_UNSUPPORTED, "qr_mask_loss_static: S = %d masks x D = %d channels need %zu bytes of scratch, the static array holds "
                                        "%d (S <= %d at D = 512): use qr_mask_loss with a workspace of your own",
                    S, D, need, QR_STATIC_SCRATCH_BYTES, QR_STATIC_MAX_MASKS);
    if (!map || !mask_id || !targets || !loss || !loss_per_mask || !d_map) return fail(QR_ERR_NULL_POINTER, "qr_mask_loss_static: NULL argument");
    if (!aligned16(map) || !aligned16(d_map)) return fail(QR_ERR_MISALIGNED, "qr_mask_loss_static: map / d_map must be 16-byte aligned");
    void* ws = nullptr;
    if (int rc = static_scratch_ptr(&ws)) return rc;
    const MaskWs w = mask_ws(ws, S, D);
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t P = (int64_t)cam->width * cam->height;
    QR_CUDA_OK(cudaMemsetAsync(ws, 0, w.total, st));                 // the array keeps the last call's sums: they must start at zero
    QR_CUDA_OK(cudaMemsetAsync(loss, 0, sizeof(float), st));
    const int64_t strips = (P + kPoolStrip - 1) / kPoolStrip;
    mask_pool_kernel<<<(unsigned)((strips + 7) / 8), 256, 0, st>>>(P, D, S, map, mask_id, w.sum, w.cnt);
    QR_LAUNCH_OK("mask_pool_kernel");
    mask_mean_kernel<<<(unsigned)S, 256, 0, st>>>(D, w.sum, w.cnt, w.valid, w.norm);
    QR_LAUNCH_OK("mask_mean_kernel");
    const size_t smem = ((size_t)D + 3 * (size_t)S) * 4;
    mask_grad_kernel<<<(unsigned)S, 256, smem, st>>>(D, S, targets, w.sum, w.cnt, w.valid, w.norm, loss, loss_per_mask);
    QR_LAUNCH_OK("mask_grad_kernel");
    mask_dmap_kernel<<<(unsigned)(sm_count() * 8), 256, 0, st>>>(P, D, S, mask_id, w.sum, d_map);
    QR_LAUNCH_OK("mask_dmap_kernel");
    return QR_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// The loss fused with the render path ("would let qr_forward / qr_backward skip the 629 MB map
// round-trip").  Rendering is linear in the features and the loss pools the map by a MEAN over each mask, so
//     pooled_s = (1 / |m_s|) sum_{p in m_s} f~(p) = (1 / |m_s|) sum_i A[i,s] F[i,:],   A[i,s] = sum_{p in m_s} w^_{p,i}
//     dL/dF[i,:] = sum_p w^_{p,i} dL/dmap[p,:] = sum_s A[i,s] g_s,                      g_s = dL/dmap of every pixel of m_s
// i.e. both directions need only the small matrix A (selected Gaussians x masks), which the walk's selection lists give
// per half tile, and neither the map nor dL/dmap has to exist.  pooled_lists_kernel builds, per 16x8 half tile, A restricted
// to the half tile's union (columns) and the masks present in its 128 pixels (a handful), in shared memory, and then either
// accumulates the pooled sums (FWD: one feature row read per column, from L2) or scatters the gradient (BWD: one 16-byte
// vector reduction per thread and column, the same atomics the tcgen05 backward's epilogue issues).
// ---------------------------------------------------------------------------------------------------------------
#include "qr_sel.cuh"

namespace qr {

__device__ __forceinline__ void nb_red(float* dst, float v) { asm volatile("red.global.add.f32 [%0], %1;" ::"l"(dst), "f"(v) : "memory"); }
// four consecutive floats in one vector reduction (16-byte aligned destination)
__device__ __forceinline__ void nb_red4(float* dst, float4 v)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

constexpr int kPlThreads = 128;
constexpr int kPlMasks = 8;              // masks per round
constexpr int kPlCols = 256;             // union columns per chunk
constexpr float kPlFix = 16777216.0f;     // 2^24: weights are accumulated as 32-bit fixed point (see Ahi)

template <bool BWD>
__global__ void __launch_bounds__(kPlThreads) pooled_lists_kernel(const Cam cam, const int K, const int D, const int S, const int64_t N,
                                                                  const SelLists sl, const int32_t* __restrict__ mask_id,
                                                                  const float* __restrict__ features, float* __restrict__ sum,
                                                                  int32_t* __restrict__ cnt, const float* __restrict__ g,
                                                                  float* __restrict__ dL_dfeat)
{
    // A is accumulated with NATIVE 32-bit integer shared-memory atomics on weights scaled by 2^24 (float and 64-bit atomicAdd on
    // shared memory are compare-and-swap loops, and ~37 entries hit each cell: half of this kernel's instructions), then
    // converted.  A cell sums at most 128 weights <= 1: 2^31 fits; the rounding, 2^-25 per entry, is far inside the tolerance.
    __shared__ uint32_t Ahi[kPlMasks][kPlCols];
    __shared__ float Ah[kPlMasks][kPlCols];
    __shared__ int32_t hkey[256];            // tiny hash set: mask id -> local index
    __shared__ int32_t hloc[256];
    __shared__ int32_t loc_mask[kHalfPx];    // local index -> mask id
    __shared__ uint8_t px_loc[kHalfPx];      // pixel -> local mask index (255: none)
    __shared__ int32_t nm_s;
    __shared__ int32_t uid_s[kPlCols];       // the chunk's union ids, staged once (a per-column global load chain cost 1 us per column)
    __shared__ __align__(16) float gs[BWD ? kPlMasks * QR_MAX_D : 4];
    if (!sel_stamp_ok(sl.stamp, cam, K)) return;
    const int tid = threadIdx.x;
    const int ht = blockIdx.x, tile = ht >> 1;
    const int x0 = (tile % cam.tiles_x) * kTile, y0 = (tile / cam.tiles_x) * kTile + (ht & 1) * 8;
    if (y0 >= cam.height) return;
    const int32_t* hdr = sl.hdr + (size_t)ht * kHdrWords;
    const int U = hdr[4];
    const int n0 = hdr[0], n1 = hdr[1], n2 = hdr[2], n3 = hdr[3];
    // masks present in the half tile, numbered locally
    for (int i = tid; i < 256; i += kPlThreads) hkey[i] = -1;
    if (tid == 0) nm_s = 0;
    __syncthreads();
    {
        const int px = x0 + (tid & 15), py = y0 + (tid >> 4);
        int m = -1;
        if (px < cam.width && py < cam.height) m = mask_id[(int64_t)py * cam.width + px];
        if (m < 0 || m >= S) m = -1;
        int loc = 255;
        // one representative per (warp, mask) inserts: masks are spatially coherent, a warp usually holds one or two
        const uint32_t peers = __match_any_sync(0xffffffffu, m);
        const bool leader = (int)(__ffs(peers) - 1) == (tid & 31);
        if (m >= 0) {
            if (!BWD && leader) atomicAdd(cnt + m, __popc(peers));
            uint32_t h = hash32((uint32_t)m) & 255u;
            if (leader) {
                while (true) {
                    const int old = atomicCAS(&hkey[h], -1, m);
                    if (old == -1) { const int l = atomicAdd(&nm_s, 1); hloc[h] = l; loc_mask[l] = m; break; }
                    if (old == m) break;
                    h = (h + 1) & 255u;
                }
            }
            h = __shfl_sync(peers, h, __ffs(peers) - 1);
            loc = (int)h;
        }
        __syncthreads();
        px_loc[tid] = m >= 0 ? (uint8_t)hloc[loc] : (uint8_t)255;
    }
    __syncthreads();
    const int nm = nm_s;
    if (U == 0 || nm == 0) return;
    const uint2* ent = sl.ent + (size_t)ht * kSelLists * sl.qcap;
    const int32_t* uid = sl.uid + (size_t)ht * sl.ucap;
    const int nl[4] = { n0, n1, n2, n3 };
    const int d4 = D >> 2;
    for (int m0 = 0; m0 < nm; m0 += kPlMasks) {
        const int nmr = min(kPlMasks, nm - m0);
        if (BWD) {          // gradient rows of this round's masks
            for (int i = tid; i < nmr * d4; i += kPlThreads) {
                const int l = i / d4, c4 = i - l * d4;
                reinterpret_cast<float4*>(gs + l * QR_MAX_D)[c4] = __ldg(reinterpret_cast<const float4*>(g + (int64_t)loc_mask[m0 + l] * D) + c4);
            }
        }
        for (int c0 = 0; c0 < U; c0 += kPlCols) {
            const int nc = min(kPlCols, U - c0);
            for (int i = tid; i < kPlMasks * kPlCols; i += kPlThreads) (&Ahi[0][0])[i] = 0u;
            for (int i = tid; i < nc; i += kPlThreads) uid_s[i] = __ldg(uid + c0 + i);
            __syncthreads();
            for (int q = 0; q < kSelLists; ++q) {              // A[col, mask] += w over the half tile's entries
                const uint2* lq = ent + (size_t)q * sl.qcap;
                // consecutive entries of a list are the pixels that selected ONE Gaussian (one column) at one walk step, so a warp's 32
                // entries fall into a few cells: sum each cell's group with one REDUX and let its first lane do the atomic
                for (int i0 = (tid & ~31); i0 < nl[q]; i0 += kPlThreads) {
                    const int i = i0 + (tid & 31);
                    int cell = -1;
                    uint32_t fx = 0u;
                    if (i < nl[q]) {
                        const uint2 e = __ldg(lq + i);
                        const int col = sel_col(e.y) - c0;
                        const int l = (int)px_loc[sel_pixel(e.y)] - m0;
                        if (col >= 0 && col < nc && l >= 0 && l < nmr) { cell = l * kPlCols + col; fx = __float2uint_rn(__uint_as_float(e.x) * kPlFix); }
                    }
                    uint32_t todo = __ballot_sync(0xffffffffu, cell >= 0);
                    while (todo) {
                        const int key = __shfl_sync(0xffffffffu, cell, __ffs(todo) - 1);
                        const uint32_t grp = __ballot_sync(0xffffffffu, cell == key);
                        const uint32_t sum = __reduce_add_sync(0xffffffffu, cell == key ? fx : 0u);
                        if ((int)(__ffs(grp) - 1) == (tid & 31)) atomicAdd(&(&Ahi[0][0])[key], sum);
                        todo &= ~grp;
                    }
                }
            }
            __syncthreads();
            for (int i = tid; i < kPlMasks * kPlCols; i += kPlThreads) (&Ah[0][0])[i] = (float)(&Ahi[0][0])[i] * (1.0f / kPlFix);
            __syncthreads();
            if (tid < d4) {
                if (!BWD) {
                    float4 acc[kPlMasks];
#pragma unroll
                    for (int l = 0; l < kPlMasks; ++l) acc[l] = make_float4(0.f, 0.f, 0.f, 0.f);
                    for (int col0 = 0; col0 < nc; col0 += 4) {           // four feature rows in flight
                        float4 f[4];
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            const int col = min(col0 + u, nc - 1);
                            f[u] = __ldg(reinterpret_cast<const float4*>(features + (int64_t)uid_s[col] * D) + tid);
                        }
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            if (col0 + u < nc) {
#pragma unroll
                                for (int l = 0; l < kPlMasks; ++l) {
                                    const float a = Ah[l][col0 + u];
                                    acc[l].x = fmaf(a, f[u].x, acc[l].x); acc[l].y = fmaf(a, f[u].y, acc[l].y);
                                    acc[l].z = fmaf(a, f[u].z, acc[l].z); acc[l].w = fmaf(a, f[u].w, acc[l].w);
                                }
                            }
                        }
                    }
#pragma unroll
                    for (int l = 0; l < kPlMasks; ++l) {
                        if (l < nmr) {
                            float* dst = sum + (int64_t)loc_mask[m0 + l] * D + 4 * tid;
                            nb_red4(dst, acc[l]);
                        }
                    }
                } else {
                    for (int col = 0; col < nc; ++col) {
                        float4 d = make_float4(0.f, 0.f, 0.f, 0.f);
                        bool any = false;
#pragma unroll
                        for (int l = 0; l < kPlMasks; ++l) {
                            const float a = Ah[l][col];
                            if (l < nmr && a != 0.0f) {
                                const float4 gv = reinterpret_cast<const float4*>(gs + l * QR_MAX_D)[tid];
                                d.x = fmaf(a, gv.x, d.x); d.y = fmaf(a, gv.y, d.y); d.z = fmaf(a, gv.z, d.z); d.w = fmaf(a, gv.w, d.w);
                                any = true;
                            }
                        }
                        if (!any) continue;
                        const int32_t id = uid_s[col];
                        if ((uint32_t)id >= (uint32_t)N) continue;      // never add outside the table
                        float* dst = dL_dfeat + (int64_t)id * D + 4 * tid;
                        nb_red4(dst, d);
                    }
                }
            }
            __syncthreads();
        }
    }
}

}  // namespace qr

extern "C" int qr_pooled_loss(const qr_camera* cam, int32_t K, int32_t D, int64_t N, void* fwd_ws, size_t fwd_ws_bytes,
                              const float* features, const int32_t* mask_id, int32_t S, const float* targets, float* loss,
                              float* loss_per_mask, float* dL_dfeat, void* ws, size_t ws_bytes, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (K < 1 || K > QR_MAX_K) return fail(QR_ERR_INVALID_ARG, "qr_pooled_loss: K out of range");
    if (!tc_channels_supported(D) || D > kNbMaxC)
        return fail(QR_ERR_UNSUPPORTED, "qr_pooled_loss: needs fp32 features on a shape of the tcgen05 path (D %% 32 == 0, or D < 32 with D %% 4 == 0; D = %d)", D);
    if (S < 1 || S > QR_MAX_MASKS) return fail(QR_ERR_INVALID_ARG, "qr_pooled_loss: S = %d outside [1, QR_MAX_MASKS]", S);
    if (N < 1) return fail(QR_ERR_INVALID_ARG, "qr_pooled_loss: N < 1");
    if (!fwd_ws || !features || !mask_id || !targets || !loss || !loss_per_mask || !ws) return fail(QR_ERR_NULL_POINTER, "qr_pooled_loss: NULL argument");
    if (!aligned16(features) || !aligned16(fwd_ws) || !aligned16(ws) || (dL_dfeat && !aligned16(dL_dfeat)))
        return fail(QR_ERR_MISALIGNED, "qr_pooled_loss: 16-byte alignment");
    const Cam c = make_cam(cam);
    const WsLayout wl = ws_layout(c, K);
    if (fwd_ws_bytes < wl.total) return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_pooled_loss: forward workspace %zu < %zu bytes", fwd_ws_bytes, wl.total);
    const MaskWs w = mask_ws(ws, S, D);
    if (ws_bytes < w.total) return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_pooled_loss: workspace %zu < %zu bytes", ws_bytes, w.total);
    const SelLists sl = sel_view(wl.sel, fwd_ws);
    cudaStream_t st = (cudaStream_t)stream;
    const unsigned nh = (unsigned)(c.tiles_x * c.tiles_y * 2);
    QR_CUDA_OK(cudaMemsetAsync(ws, 0, w.total, st));
    QR_CUDA_OK(cudaMemsetAsync(loss, 0, sizeof(float), st));
    pooled_lists_kernel<false><<<nh, kPlThreads, 0, st>>>(c, K, D, S, N, sl, mask_id, features, w.sum, w.cnt, nullptr, nullptr);
    QR_LAUNCH_OK("pooled_lists_kernel<fwd>");
    mask_mean_kernel<<<(unsigned)S, 256, 0, st>>>(D, w.sum, w.cnt, w.valid, w.norm);
    QR_LAUNCH_OK("mask_mean_kernel");
    const size_t smem = ((size_t)D + 3 * (size_t)S) * 4;
    mask_grad_kernel<<<(unsigned)S, 256, smem, st>>>(D, S, targets, w.sum, w.cnt, w.valid, w.norm, loss, loss_per_mask);
    QR_LAUNCH_OK("mask_grad_kernel");
    if (dL_dfeat) {
        pooled_lists_kernel<true><<<nh, kPlThreads, 0, st>>>(c, K, D, S, N, sl, mask_id, features, nullptr, nullptr, w.sum, dL_dfeat);
        QR_LAUNCH_OK("pooled_lists_kernel<bwd>");
    }
    return QR_OK;
}

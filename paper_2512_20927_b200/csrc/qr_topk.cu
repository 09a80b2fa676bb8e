// qr_topk.cu -- qr_topk_forward: the paper's other comparator, top-K render ("top-K sampling proposed by a
// concurrent study, which requires additional complexity to sort values, O(N log K + KC)"; complexity table
// PAPER.md:187; speed / accuracy figure).  The paper gives no procedure; this follows the
// reconstruction of SPEC.md:221-229 (reading R17):
//   1. dense weights of Eq. 1, w = T alpha', over the pixel's list, with V-Render's early stop R7;
//   2. keep the K largest (ties -> the earlier list position);
//   3. re-blend the kept entries in depth order with a fresh transmittance;  4. normalise by 1 - T^top (line 20).
//
// topk_select_kernel is the O(N log K) part: CTA = 16x8 half tile, thread = pixel.  The tile's list is staged 128 entries at
// a time; every thread evaluates alpha' (rule R4, the fp32 decision arithmetic of DESIGN.md), carries the dense T and
// keeps the K largest weights in a binary min-heap in shared memory, ordered by (weight, later position first) so that
// the root is always the entry to drop.  After the walk the heap is sorted by list position (depth order), re-blended
// and written as selection records (sel_idx, sel_w, n_sel, resid) in qr_forward's format: qr_backward accepts them.
//
// The O(KC) part is the SAME contraction as Q-Render's: for fp32 features with D % 128 == 0 backward_prep_kernel numbers
// each half tile's union and writes the entry lists, and blend_mma_kernel (tcgen05) blends them; half tiles with more
// records than the prep takes, and every other shape, go through records_blend_kernel (one warp per pixel, the plain
// statement of  out[p,:] = sum_s sel_w[p,s] F[sel_idx[p,s],:]).
#include "qr_backward.cuh"
#include "qr_blend.cuh"

namespace qr {

constexpr int kTkThreads = 128;          // CTA = one 16x8-pixel half tile, thread = pixel
constexpr int kTkBatch = 128;

struct TopkParams {
    Cam cam;
    int32_t K;
    float t_min;
    const float2* mean2d;
    const float4* conic_opac;
    const uint32_t* isect;
    const int2* tile_range;
    int32_t* n_sel;
    float* resid;
    int32_t* sel_idx;
    float* sel_w;
};

// (w1, pos1) is dropped before (w2, pos2): the smaller weight; among equal weights the later list position
__device__ __forceinline__ bool tk_less(float w1, int p1, float w2, int p2) { return w1 < w2 || (w1 == w2 && p1 > p2); }

// alpha' of a Gaussian at a pixel centre with inclusion rule R4 (0 = not in the pixel's list), the operation order of DESIGN.md 2
__device__ __forceinline__ float tk_alpha(float fpx, float fpy, float2 xy, float4 co)
{
    const float dx = __fsub_rn(fpx, xy.x), dy = __fsub_rn(fpy, xy.y);
    const float q1 = __fmul_rn(__fmul_rn(co.x, dx), dx);
    const float q2 = __fmaf_rn(__fmul_rn(co.z, dy), dy, q1);
    const float q3 = __fmul_rn(__fmul_rn(co.y, dx), dy);
    const float power = __fmaf_rn(-0.5f, q2, -q3);
    if (power > 0.0f || power < kPowerMin) return 0.0f;
    const float a = fminf(kAlphaMax, __fmul_rn(co.w, expf(power)));
    return a < kAlphaMin ? 0.0f : a;
}

// The heap lives in SHARED memory, slot-major ([slot][thread]: conflict free), and holds only (weight, list position): 8 K
// bytes per pixel.  (The first version kept {w, alpha', id, pos} per thread in local memory: 1 KB x 256 threads x 8 CTAs per SM
// thrashed L1 and the kernel took 1.8 ms at config 3.)  alpha' and the id of the kept entries are recomputed from their list
// positions after the walk -- the same arithmetic on the same inputs, so the same bits.
__global__ void __launch_bounds__(kTkThreads) topk_select_kernel(const TopkParams p)
{
    extern __shared__ __align__(16) unsigned char tk_smem[];
    __shared__ float4 s_co[kTkBatch];
    __shared__ float2 s_xy[kTkBatch];
    const int tid = threadIdx.x;
    const int K = p.K;
    float* hw = reinterpret_cast<float*>(tk_smem) + tid;                  // hw[i * kTkThreads]
    int32_t* hp = reinterpret_cast<int32_t*>(tk_smem) + K * kTkThreads + tid;
    const int ht = blockIdx.x, tile = ht >> 1;
    const int x0 = (tile % p.cam.tiles_x) * kTile, y0 = (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8;
    const int px = x0 + (tid & 15), py = y0 + (tid >> 4);
    const bool inside = px < p.cam.width && py < p.cam.height;
    const float fpx = (float)px + 0.5f, fpy = (float)py + 0.5f;          // R5
    const int2 range = p.tile_range[tile];
#define HW(i) hw[(i) * kTkThreads]
#define HP(i) hp[(i) * kTkThreads]
    int nh = 0;
    float T = 1.0f;
    bool done = !inside;

    for (int b0 = range.x; b0 < range.y; b0 += kTkBatch) {
        if (__syncthreads_and(done)) break;
        {
            const int idx = b0 + tid;
            float4 co = make_float4(0.f, 0.f, 0.f, 0.f);
            float2 xy = make_float2(0.f, 0.f);
            if (idx < range.y) { const int32_t id = (int32_t)p.isect[idx]; xy = __ldg(p.mean2d + id); co = __ldg(p.conic_opac + id); }
            s_xy[tid] = xy; s_co[tid] = co;
        }
        __syncthreads();
        if (done) continue;
        const int nb = min(kTkBatch, range.y - b0);
        for (int e = 0; e < nb; ++e) {
            const float a = tk_alpha(fpx, fpy, s_xy[e], s_co[e]);
            if (a == 0.0f) continue;
            const float T_test = __fmul_rn(T, __fsub_rn(1.0f, a));
            if (T_test < p.t_min) { done = true; break; }                 // R7: stop WITHOUT this entry
            const float w = __fmul_rn(T, a);                              // Eq. 1 weight (step 1)
            const int pos = b0 - range.x + e;
            if (nh < K) {                                                 // step 2: K largest, min-heap
                int i = nh++;
                while (i > 0) {
                    const int par = (i - 1) >> 1;
                    const float pw = HW(par); const int pp = HP(par);
                    if (!tk_less(w, pos, pw, pp)) break;
                    HW(i) = pw; HP(i) = pp;
                    i = par;
                }
                HW(i) = w; HP(i) = pos;
            } else if (w > HW(0)) {                                       // equal to the smallest kept: the earlier one stays
                int i = 0;
                while (true) {
                    int c = 2 * i + 1;
                    if (c >= nh) break;
                    float cw = HW(c); int cp = HP(c);
                    if (c + 1 < nh) {
                        const float cw2 = HW(c + 1); const int cp2 = HP(c + 1);
                        if (tk_less(cw2, cp2, cw, cp)) { ++c; cw = cw2; cp = cp2; }
                    }
                    if (!tk_less(cw, cp, w, pos)) break;
                    HW(i) = cw; HP(i) = cp;
                    i = c;
                }
                HW(i) = w; HP(i) = pos;
            }
            T = T_test;
        }
    }
    if (!inside) return;
    // depth order = list position (insertion sort on the positions; K <= 64)
    for (int i = 1; i < nh; ++i) {
        const int pos = HP(i);
        int j = i - 1;
        while (j >= 0 && HP(j) > pos) { HP(j + 1) = HP(j); --j; }
        HP(j + 1) = pos;
    }
    // steps 3, 4: fresh transmittance over the kept entries in depth order, then normalise
    const int64_t pix = (int64_t)py * p.cam.width + px;
    float Tt = 1.0f;
    for (int i = 0; i < nh; ++i) {
        const int32_t id = (int32_t)p.isect[range.x + HP(i)];
        const float a = tk_alpha(fpx, fpy, __ldg(p.mean2d + id), __ldg(p.conic_opac + id));
        HW(i) = __fmul_rn(Tt, a);
        Tt = __fmul_rn(Tt, __fsub_rn(1.0f, a));
        p.sel_idx[pix * K + i] = id;
    }
    const float inv = nh > 0 ? __fdiv_rn(1.0f, __fsub_rn(1.0f, Tt)) : 0.0f;
    for (int i = 0; i < nh; ++i) p.sel_w[pix * K + i] = __fmul_rn(HW(i), inv);
    p.n_sel[pix] = nh;
    p.resid[pix] = nh > 0 ? Tt : 1.0f;                                    // R8
#undef HW
#undef HP
}

__device__ __forceinline__ float tk_f32(float v) { return v; }
__device__ __forceinline__ float tk_f32(__half v) { return __half2float(v); }

// out[p,:] = sum_s sel_w[p,s] F[sel_idx[p,s],:]   -- one warp per pixel, lane c of every 32-channel group.
// hdr != nullptr: only the pixels of half tiles whose header carries the "left over" flag (hdr[5] == 1).
template <typename FeatT>
__global__ void __launch_bounds__(256) records_blend_kernel(const Cam cam, const int K, const int D, const FeatT* __restrict__ features,
                                                            const int32_t* __restrict__ sel_idx, const float* __restrict__ sel_w,
                                                            const int32_t* __restrict__ n_sel, float* __restrict__ out_map,
                                                            const int32_t* __restrict__ hdr, const int32_t* __restrict__ nflag)
{
    if (nflag && *nflag == 0) return;
    const int lane = threadIdx.x & 31;
    const int64_t npix = (int64_t)cam.width * cam.height;
    const int64_t warps = (int64_t)gridDim.x * (blockDim.x >> 5);
    for (int64_t pix = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); pix < npix; pix += warps) {
        if (hdr) {
            const int x = (int)(pix % cam.width), y = (int)(pix / cam.width);
            const int ht = ((y >> 4) * cam.tiles_x + (x >> 4)) * 2 + ((y >> 3) & 1);
            if (hdr[(size_t)ht * kHdrWords + 5] != 1) continue;
        }
        const int n = max(0, min(K, n_sel[pix]));
        float acc[QR_MAX_D / 32];
#pragma unroll
        for (int j = 0; j < QR_MAX_D / 32; ++j) acc[j] = 0.0f;
        for (int s = 0; s < n; ++s) {
            const int32_t id = sel_idx[pix * K + s];
            const float w = sel_w[pix * K + s];
            const FeatT* row = features + (int64_t)id * D;
#pragma unroll
            for (int j = 0; j < QR_MAX_D / 32; ++j) {
                const int c = j * 32 + lane;
                if (c < D) acc[j] = __fmaf_rn(w, tk_f32(row[c]), acc[j]);
            }
        }
        float* o = out_map + pix * D;
#pragma unroll
        for (int j = 0; j < QR_MAX_D / 32; ++j) {
            const int c = j * 32 + lane;
            if (c < D) o[c] = acc[j];
        }
    }
}

}  // namespace qr

extern "C" size_t qr_topk_workspace_bytes(const qr_camera* cam, int32_t K, int32_t D)
{
    if (!cam || cam->width < 1 || cam->height < 1 || K < 1 || K > QR_TOPK_MAX_K) return 0;
    if (qr::tc_channels_supported(D)) return qr::ws_layout(qr::make_cam(cam), K).total;
    return 256;
}

extern "C" int qr_topk_forward(const qr_camera* cam, int32_t K, int32_t D, qr_dtype feat_dtype, float t_min,
                               const float* mean2d, const float* conic_opac, const uint32_t* isect_gauss,
                               const int32_t* tile_range, const void* features, float* out_map, int32_t* sel_idx,
                               float* sel_w, int32_t* n_sel, float* resid, void* ws, size_t ws_bytes, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (K < 1) return fail(QR_ERR_INVALID_ARG, "qr_topk_forward: K = %d < 1 (SPEC.md:226)", K);
    if (K > QR_TOPK_MAX_K) return fail(QR_ERR_UNSUPPORTED, "qr_topk_forward: K = %d > QR_TOPK_MAX_K", K);
    if (int rc = check_feat(D, feat_dtype, "qr_topk_forward")) return rc;
    if (!(t_min >= 0.0f)) return fail(QR_ERR_INVALID_ARG, "qr_topk_forward: t_min must be >= 0");
    if (!mean2d || !conic_opac || !isect_gauss || !tile_range || !features || !out_map || !sel_idx || !sel_w || !n_sel || !resid)
        return fail(QR_ERR_NULL_POINTER, "qr_topk_forward: NULL argument");
    if (!aligned16(out_map) || !aligned16(features) || !aligned16(conic_opac) || !aligned16(mean2d))
        return fail(QR_ERR_MISALIGNED, "qr_topk_forward: out_map / features / conic_opac / mean2d must be 16-byte aligned");
    const Cam c = make_cam(cam);
    cudaStream_t st = (cudaStream_t)stream;
    const int T = c.tiles_x * c.tiles_y;

    TopkParams tp;
    tp.cam = c; tp.K = K; tp.t_min = t_min;
    tp.mean2d = reinterpret_cast<const float2*>(mean2d);
    tp.conic_opac = reinterpret_cast<const float4*>(conic_opac);
    tp.isect = isect_gauss; tp.tile_range = reinterpret_cast<const int2*>(tile_range);
    tp.n_sel = n_sel; tp.resid = resid; tp.sel_idx = sel_idx; tp.sel_w = sel_w;
    const size_t heap_bytes = (size_t)K * kTkThreads * 8;                  // <= 64 KB at K = 64
    QR_CUDA_OK(cudaFuncSetAttribute(topk_select_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)heap_bytes));
    topk_select_kernel<<<(unsigned)T * 2u, kTkThreads, heap_bytes, st>>>(tp);
    QR_LAUNCH_OK("topk_select_kernel");

    const int sms = sm_count();
    const unsigned rgrid = (unsigned)(sms * 8);
    const bool mma = blend_mma_supported(D, feat_dtype);
    if (mma) {
        const WsLayout wl = ws_layout(c, K);
        if (!ws) return fail(QR_ERR_NULL_POINTER, "qr_topk_forward: workspace is NULL");
        if (ws_bytes < wl.total) return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_topk_forward: workspace %zu < %zu bytes", ws_bytes, wl.total);
        if (!aligned16(ws)) return fail(QR_ERR_MISALIGNED, "qr_topk_forward: workspace alignment");
        BackwardParams bp;
        bp.cam = c; bp.K = K; bp.D = D; bp.N = 0;
        bp.sel_idx = sel_idx; bp.sel_w = sel_w; bp.n_sel = n_sel; bp.dL_dmap = nullptr; bp.dL_dfeat = nullptr;
        bp.sl = sel_view(wl.sel, ws);
        int32_t* nflag = reinterpret_cast<int32_t*>(ws);
        QR_CUDA_OK(cudaMemsetAsync(nflag, 0, 256, st));
        // the blend's ticket = 0, every half tile's ready flag != 0 (the lists are complete when the blend starts)
        QR_CUDA_OK(cudaMemsetAsync(bp.sl.ctrl, 0, (size_t)kCtrlWords * 4, st));
        QR_CUDA_OK(cudaMemsetAsync(bp.sl.flags, 1, (size_t)T * 2 * 4, st));
        if (int rc = launch_backward_prep(bp, nflag, st)) return rc;
        BlendParams bl;
        bl.cam = c; bl.K = K; bl.D = D; bl.cap = 0; bl.num_tiles = T; bl.tile_ticket = nullptr;
        bl.features = features; bl.gcount = nullptr; bl.ucount = nullptr; bl.rec = nullptr;
        bl.n_sel = n_sel; bl.resid = resid; bl.out_map = out_map; bl.sel_idx = sel_idx; bl.sel_w = sel_w;
        bl.sl = bp.sl;
        bl.feat_f16 = feat_dtype == QR_F16 ? 1 : 0;
        if (int rc = launch_blend_mma(bl, st, false)) return rc;
        if (feat_dtype == QR_F16)
            records_blend_kernel<__half><<<rgrid, 256, 0, st>>>(c, K, D, static_cast<const __half*>(features), sel_idx, sel_w, n_sel,
                                                                out_map, bp.sl.hdr, nflag);
        else
            records_blend_kernel<float><<<rgrid, 256, 0, st>>>(c, K, D, static_cast<const float*>(features), sel_idx, sel_w, n_sel,
                                                               out_map, bp.sl.hdr, nflag);
        QR_LAUNCH_OK("records_blend_kernel");
        return QR_OK;
    }
    if (feat_dtype == QR_F16)
        records_blend_kernel<__half><<<rgrid, 256, 0, st>>>(c, K, D, static_cast<const __half*>(features), sel_idx, sel_w, n_sel,
                                                            out_map, nullptr, nullptr);
    else
        records_blend_kernel<float><<<rgrid, 256, 0, st>>>(c, K, D, static_cast<const float*>(features), sel_idx, sel_w, n_sel,
                                                           out_map, nullptr, nullptr);
    QR_LAUNCH_OK("records_blend_kernel");
    return QR_OK;
}

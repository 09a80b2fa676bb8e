// qr_render.cu -- qr_dense_forward (Eq. 1), the in-run dense comparator, as a fused band kernel (the FFMA
// formulation: the first fused design of this build, kept for the comparator; Q-Render itself lives in qr_walk.cu,
// qr_blend_mma.cu and qr_forward.cu).
//
// Work decomposition:
//   CTA  = one 16x4-pixel band of a 16x16 tile (4 CTAs share a tile's depth-sorted list), 256 threads = 8 warps.
//   The tile list is consumed in batches of 32 entries:
//     load     32 threads gather (id, mean2d, conic, opacity) of the batch into shared memory and derive a
//              conservative screen-space box of the 3-sigma ellipse;
//     evaluate all 8 warps: warp (h, j) tests entries j, j+4, ... against the 32 pixels of half-band h; entries whose
//              box misses the warp's pixels are skipped with one uniform branch; alpha' goes to shared memory, the
//              per-entry inclusion ballot to pmask;
//     resolve  2 warps, one thread per pixel: the sequential part of Eq. 1 (T, T_test, the early stop R7) in list order
//              over the included entries only; the weights T alpha' go to Wb, and a per pixel-group bit mask of
//              "entries some pixel of the group blends" is built with ballots;
//     blend    all 8 warps: warp g owns the 4x2-pixel group g and all D channels (lane = 4 consecutive channels per
//              128-channel slab): for every entry of its mask it loads the feature row once (128-bit coalesced,
//              L1-resident across the groups of a tile) and applies it to the 8 pixels from registers.
//   Epilogue: 128-bit streaming stores of the HWC map (no normalisation), final T per pixel.
//
// fp32 decision arithmetic (power, alpha', T) uses explicit rounding intrinsics in the order fixed in DESIGN.md; the
// library is also compiled with -fmad=false.
#include "qr_blend.cuh"
#include "qr_common.cuh"
#include "qr_sel.cuh"

namespace qr {

constexpr int kBatch = 32;           // list entries per batch
constexpr int kBandH = 4;            // pixel rows per CTA
constexpr int kBandPx = kTile * kBandH;   // 64 pixels per CTA
constexpr int kGroups = 8;           // 4x2-pixel groups per band
constexpr int kRenderThreads = 256;

struct RenderParams {
    Cam cam;
    int32_t D;
    float t_min;
    const float2* mean2d;
    const float4* conic_opac;
    const uint32_t* isect;
    const int2* tile_range;
    const void* features;
    float* out_map;
    float* final_T;
    const int32_t* only_hdr = nullptr;   // qr_dense_forward_tc: headers of the selection lists; a band runs only if its half tile is flagged
};

template <typename FeatT, int VW> struct RowLoad;
template <> struct RowLoad<float, 4> {
    static __device__ __forceinline__ void load(const void* base, int64_t row, int D, int ch, float (&f)[4])
    {
        const float4 v = __ldg(reinterpret_cast<const float4*>(static_cast<const float*>(base) + row * D + ch));
        f[0] = v.x; f[1] = v.y; f[2] = v.z; f[3] = v.w;
    }
};
template <> struct RowLoad<float, 1> {
    static __device__ __forceinline__ void load(const void* base, int64_t row, int D, int ch, float (&f)[1])
    {
        f[0] = __ldg(static_cast<const float*>(base) + row * D + ch);
    }
};
template <> struct RowLoad<__half, 8> {
    static __device__ __forceinline__ void load(const void* base, int64_t row, int D, int ch, float (&f)[8])
    {
        const uint4 v = __ldg(reinterpret_cast<const uint4*>(static_cast<const __half*>(base) + row * D + ch));
        const __half2* h = reinterpret_cast<const __half2*>(&v);
#pragma unroll
        for (int i = 0; i < 4; ++i) { const float2 t = __half22float2(h[i]); f[2 * i] = t.x; f[2 * i + 1] = t.y; }
    }
};

template <int VW> __device__ __forceinline__ void store_out(float* dst, const float (&v)[VW]);
template <> __device__ __forceinline__ void store_out<4>(float* dst, const float (&v)[4])
{
    __stcs(reinterpret_cast<float4*>(dst), make_float4(v[0], v[1], v[2], v[3]));
}
template <> __device__ __forceinline__ void store_out<1>(float* dst, const float (&v)[1]) { __stcs(dst, v[0]); }
template <> __device__ __forceinline__ void store_out<8>(float* dst, const float (&v)[8])
{
    __stcs(reinterpret_cast<float4*>(dst), make_float4(v[0], v[1], v[2], v[3]));
    __stcs(reinterpret_cast<float4*>(dst) + 1, make_float4(v[4], v[5], v[6], v[7]));
}

template <typename FeatT, int NV, int VW>
__global__ void __launch_bounds__(kRenderThreads, 1) render_kernel(const RenderParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // ---- shared memory carve-up ----
    float4* ent_co = reinterpret_cast<float4*>(smem_raw);                       // [32] a, b, c, opacity
    float4* ent_box = ent_co + kBatch;                                          // [32] x_lo, x_hi, y_lo, y_hi
    float2* ent_xy = reinterpret_cast<float2*>(ent_box + kBatch);               // [32]
    int32_t* ent_id = reinterpret_cast<int32_t*>(ent_xy + kBatch);              // [32]
    uint32_t* pmask = reinterpret_cast<uint32_t*>(ent_id + kBatch);             // [32][2]
    uint32_t* gmask = pmask + 2 * kBatch;                                       // [8]
    uint32_t* done_mask = gmask + kGroups;                                      // [2]
    float* A = reinterpret_cast<float*>(done_mask + 4);                         // [32][64] alpha' (2 + 2 pad words: 16-byte aligned)
    float* Wb = A + kBatch * kBandPx;                                           // [32][64] blending weights
    const int D = p.D;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x >> 2, band = blockIdx.x & 3;
    const int tile_x = tile % p.cam.tiles_x, tile_y = tile / p.cam.tiles_x;
    const int x0 = tile_x * kTile, y0 = tile_y * kTile + band * kBandH;
    if (y0 >= p.cam.height) return;   // band entirely below the image
    if (p.only_hdr && p.only_hdr[(size_t)(tile * 2 + (band >> 1)) * kHdrWords + 5] != 1) return;    // not left to this kernel

    // ---- init ----
    for (int i = tid; i < kBatch * kBandPx; i += kRenderThreads) Wb[i] = 0.0f;
    const int2 range = p.tile_range[tile];

    // resolve state (meaningful in warps 0, 1 only: thread = pixel)
    const int rp = tid;                                  // local pixel index when tid < 64
    const int rpx = x0 + (rp & 15), rpy = y0 + ((rp >> 4) & 3);
    bool done = !(tid < kBandPx && rpx < p.cam.width && rpy < p.cam.height);
    float T = 1.0f;
    const float t_break = p.t_min;
    if (tid < kBandPx) {
        const uint32_t dm = __ballot_sync(0xffffffffu, done);
        if (lane == 0) done_mask[warp] = dm;
    }

    // evaluate role: half-band h, entry slot j
    const int eh = warp & 1, ej = warp >> 1;
    const int epx = x0 + (lane & 15), epy = y0 + eh * 2 + (lane >> 4);
    const float fpx = (float)epx + 0.5f, fpy = (float)epy + 0.5f;     // R5
    const float wx_lo = (float)x0, wx_hi = (float)(x0 + kTile);        // pixel-centre range of this warp is inside
    const float wy_lo = (float)(y0 + eh * 2), wy_hi = (float)(y0 + eh * 2 + 2);

    // blend role: group g = warp
    const int gx = warp & 3, gy = warp >> 2;
    float acc[8][NV][VW];
#pragma unroll
    for (int q = 0; q < 8; ++q)
#pragma unroll
        for (int j = 0; j < NV; ++j)
#pragma unroll
            for (int v = 0; v < VW; ++v) acc[q][j][v] = 0.0f;

    __syncthreads();

    for (int b0 = range.x; b0 < range.y; b0 += kBatch) {
        // ---------------- load ----------------
        if (tid < kBatch) {
            const int idx = b0 + tid;
            int32_t id = -1;
            float4 co = make_float4(0.f, 0.f, 0.f, 0.f), box = make_float4(1.f, 0.f, 1.f, 0.f);   // empty box
            float2 xy = make_float2(0.f, 0.f);
            if (idx < range.y) {
                id = (int32_t)p.isect[idx];
                xy = __ldg(p.mean2d + id);
                co = __ldg(p.conic_opac + id);
                // 3-sigma ellipse AABB from the conic: cov = conic^-1, half-widths 3 sqrt(cov_xx), 3 sqrt(cov_yy),
                // inflated so that fp32 rounding can never exclude a pixel that rule R4 includes
                const float det = co.x * co.z - co.y * co.y;
                float ex = 3.0e30f, ey = 3.0e30f;
                if (det > 0.0f) {
                    ex = 3.0f * sqrtf(co.z / det) * 1.001f + 0.01f;
                    ey = 3.0f * sqrtf(co.x / det) * 1.001f + 0.01f;
                }
                box = make_float4(xy.x - ex, xy.x + ex, xy.y - ey, xy.y + ey);
            }
            ent_id[tid] = id; ent_co[tid] = co; ent_xy[tid] = xy; ent_box[tid] = box;
        }
        __syncthreads();

        // ---------------- evaluate ----------------
        {
            const uint32_t dm = done_mask[eh];
            const bool mydone = (dm >> lane) & 1u;
#pragma unroll 2
            for (int e = ej; e < kBatch; e += 4) {
                const float4 box = ent_box[e];
                uint32_t inc_mask = 0;
                // uniform cull: the warp's pixel centres lie in (wx_lo, wx_hi) x (wy_lo, wy_hi)
                if (dm != 0xffffffffu && box.x < wx_hi && box.y > wx_lo && box.z < wy_hi && box.w > wy_lo) {
                    const float4 co = ent_co[e];
                    const float2 xy = ent_xy[e];
                    const float dx = __fsub_rn(fpx, xy.x), dy = __fsub_rn(fpy, xy.y);
                    const float q1 = __fmul_rn(__fmul_rn(co.x, dx), dx);
                    const float q2 = __fmaf_rn(__fmul_rn(co.z, dy), dy, q1);
                    const float q3 = __fmul_rn(__fmul_rn(co.y, dx), dy);
                    const float power = __fmaf_rn(-0.5f, q2, -q3);
                    bool inc = !mydone && !(power > 0.0f) && !(power < kPowerMin);
                    float a = 0.0f;
                    if (inc) {
                        a = fminf(kAlphaMax, __fmul_rn(co.w, expf(power)));
                        inc = !(a < kAlphaMin);
                    }
                    inc_mask = __ballot_sync(0xffffffffu, inc);
                    if (inc) A[e * kBandPx + eh * 32 + lane] = a;
                }
                if (lane == 0) pmask[e * 2 + eh] = inc_mask;
            }
        }
        __syncthreads();

        // ---------------- resolve (Algorithm 1 lines 3-19 / Eq. 1), warps 0 and 1 ----------------
        if (warp < 2) {
            uint32_t gm = 0;                        // lanes 0..3: entries selected by some pixel of group (warp, lane)
            const uint32_t gsel = (0xFu << (4 * (lane & 3))) | (0xFu << (16 + 4 * (lane & 3)));
            for (int e = 0; e < kBatch; ++e) {
                const uint32_t pm = pmask[e * 2 + warp];
                if (pm == 0) continue;              // uniform
                bool sel = false;
                if (((pm >> lane) & 1u) && !done) {
                    const float a = A[e * kBandPx + rp];
                    const float T_test = __fmul_rn(T, __fsub_rn(1.0f, a));          // line 5
                    if (T_test < t_break) {
                        done = true;                                            // R7: stop without blending
                    } else {
                        Wb[e * kBandPx + rp] = __fmul_rn(T, a);                 // w_i = T_i alpha'_i
                        sel = true;
                        T = T_test;
                    }
                }
                const uint32_t sm = __ballot_sync(0xffffffffu, sel);
                if (sm & gsel) gm |= 1u << e;       // used by lanes 0..3 only
            }
            if (lane < 4) gmask[warp * 4 + lane] = gm;
            const uint32_t dm = __ballot_sync(0xffffffffu, done);
            if (lane == 0) done_mask[warp] = dm;
        }
        __syncthreads();

        // ---------------- blend ----------------
        {
            uint32_t m = gmask[warp];
            while (m) {
                const int e = __ffs(m) - 1;
                m &= m - 1;
                const int64_t id = ent_id[e];
                float* wrow = Wb + e * kBandPx + gy * 32 + gx * 4;
                const float4 w0 = *reinterpret_cast<const float4*>(wrow);
                const float4 w1 = *reinterpret_cast<const float4*>(wrow + 16);
                __syncwarp();
                if (lane == 0) *reinterpret_cast<float4*>(wrow) = make_float4(0.f, 0.f, 0.f, 0.f);
                if (lane == 1) *reinterpret_cast<float4*>(wrow + 16) = make_float4(0.f, 0.f, 0.f, 0.f);
                const float w[8] = { w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w };
                float f[NV][VW];
#pragma unroll
                for (int j = 0; j < NV; ++j) {
                    const int ch = (j * 32 + lane) * VW;
                    if (ch < D) RowLoad<FeatT, VW>::load(p.features, id, D, ch, f[j]);
                    else {
#pragma unroll
                        for (int v = 0; v < VW; ++v) f[j][v] = 0.0f;
                    }
                }
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    if (w[q] != 0.0f) {             // uniform across the warp
#pragma unroll
                        for (int j = 0; j < NV; ++j)
#pragma unroll
                            for (int v = 0; v < VW; ++v) acc[q][j][v] = __fmaf_rn(w[q], f[j][v], acc[q][j][v]);
                    }
                }
            }
        }
        const bool all_done = (done_mask[0] & done_mask[1]) == 0xffffffffu;
        __syncthreads();
        if (all_done) break;
    }

    // ---------------- epilogue ----------------
    if (tid < kBandPx) {
        if (rpx < p.cam.width && rpy < p.cam.height) p.final_T[(int64_t)rpy * p.cam.width + rpx] = T;
    }

    // map: warp g writes its 8 pixels, 512 contiguous bytes per store instruction
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const int lp = gy * 32 + (q >> 2) * 16 + gx * 4 + (q & 3);
        const int px = x0 + (lp & 15), py = y0 + (lp >> 4);
        if (px < p.cam.width && py < p.cam.height) {
            float* dst = p.out_map + ((int64_t)py * p.cam.width + px) * D;
#pragma unroll
            for (int j = 0; j < NV; ++j) {
                const int ch = (j * 32 + lane) * VW;
                if (ch < D) {
                    float o[VW];
#pragma unroll
                    for (int v = 0; v < VW; ++v) o[v] = acc[q][j][v];
                    store_out<VW>(dst + ch, o);
                }
            }
        }
    }
}

static size_t render_smem_bytes()
{
    size_t b = 0;
    b += kBatch * (16 + 16 + 8 + 4);             // ent_co, ent_box, ent_xy, ent_id
    b += (2 * kBatch + kGroups + 4) * 4;         // pmask, gmask, done_mask (+ 2 pad words)
    b += 2 * kBatch * kBandPx * 4;               // A, Wb
    return b + 32;
}

template <typename FeatT, int NV, int VW>
static int launch_one(const RenderParams& p, int T, cudaStream_t st)
{
    const size_t smem = render_smem_bytes();
    auto kern = render_kernel<FeatT, NV, VW>;
    QR_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<(unsigned)T * 4u, kRenderThreads, smem, st>>>(p);
    QR_LAUNCH_OK("render_kernel");
    return QR_OK;
}

static int launch_render(const RenderParams& p, qr_dtype dt, cudaStream_t st)
{
    const int T = p.cam.tiles_x * p.cam.tiles_y;
    const int D = p.D;
    if (dt == QR_F16) {
        const int nv = (D + 255) / 256;
        if (nv == 1) return launch_one<__half, 1, 8>(p, T, st);
        return launch_one<__half, 2, 8>(p, T, st);
    }
    if (D % 4 == 0) {
        const int nv = (D + 127) / 128;
        switch (nv) {
            case 1: return launch_one<float, 1, 4>(p, T, st);
            case 2: return launch_one<float, 2, 4>(p, T, st);
            case 3: return launch_one<float, 3, 4>(p, T, st);
            default: return launch_one<float, 4, 4>(p, T, st);
        }
    }
    const int nv = (D + 31) / 32;
    switch (nv) {
        case 1: return launch_one<float, 1, 1>(p, T, st);
        case 2: return launch_one<float, 2, 1>(p, T, st);
        case 3: return launch_one<float, 3, 1>(p, T, st);
        default: return launch_one<float, 4, 1>(p, T, st);
    }
}

}  // namespace qr

extern "C" int qr_dense_forward(const qr_camera* cam, int32_t D, qr_dtype feat_dtype, float t_min, const float* mean2d,
                                const float* conic_opac, const uint32_t* isect_gauss, const int32_t* tile_range,
                                const void* features, float* out_map, float* final_T, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (int rc = check_feat(D, feat_dtype, "qr_dense_forward")) return rc;
    if (!(t_min >= 0.0f)) return fail(QR_ERR_INVALID_ARG, "qr_dense_forward: t_min must be >= 0");
    if (!tile_range || !out_map || !final_T) return fail(QR_ERR_NULL_POINTER, "qr_dense_forward: NULL output or tile_range");
    if (!aligned16(out_map) || !aligned16(features) || !aligned16(conic_opac) || !aligned16(mean2d))
        return fail(QR_ERR_MISALIGNED, "qr_dense_forward: 16-byte alignment");
    RenderParams p;
    p.cam = make_cam(cam); p.D = D; p.t_min = t_min;
    p.mean2d = reinterpret_cast<const float2*>(mean2d);
    p.conic_opac = reinterpret_cast<const float4*>(conic_opac);
    p.isect = isect_gauss; p.tile_range = reinterpret_cast<const int2*>(tile_range); p.features = features;
    p.out_map = out_map; p.final_T = final_T;
    return launch_render(p, feat_dtype, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------------------------------------------
// qr_dense_forward_tc: the same Eq. 1 on the tensor cores, so that the comparator is not an FFMA kernel measured against a
// tcgen05 one.  walk2_kernel in dense mode emits every blended (Gaussian, pixel) pair with its weight T alpha' into the
// selection-list format of qr_sel.cuh (columns = the Gaussians of the half tile's list prefix that some pixel blends), and
// blend_mma_kernel -- unchanged -- contracts W[128 px, U] with F[U, D] in rounds of 64 columns.  The lists hold `cap`
// entries per pixel on average over each 32-pixel list; a half tile that needs more is flagged by the walk and rendered
// by render_kernel afterwards (it returns at once for every other band).
// ------------------------------------------------------------------------------------------------------------------
extern "C" size_t qr_dense_workspace_bytes(const qr_camera* cam, int32_t cap)
{
    if (!cam || cam->width < 1 || cam->height < 1 || cap < 1 || cap > QR_MAX_K) return 0;
    return qr::ws_layout(qr::make_cam(cam), cap).total;
}

extern "C" int qr_dense_forward_tc(const qr_camera* cam, int32_t D, qr_dtype feat_dtype, float t_min, int32_t cap,
                                   const float* mean2d, const float* conic_opac, const uint32_t* isect_gauss,
                                   const int32_t* tile_range, const void* features, float* out_map, float* final_T,
                                   void* ws, size_t ws_bytes, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (int rc = check_feat(D, feat_dtype, "qr_dense_forward_tc")) return rc;
    if (!(t_min >= 0.0f)) return fail(QR_ERR_INVALID_ARG, "qr_dense_forward_tc: t_min must be >= 0");
    if (cap < 1 || cap > QR_MAX_K) return fail(QR_ERR_INVALID_ARG, "qr_dense_forward_tc: cap = %d outside [1, QR_MAX_K]", cap);
    if (!blend_mma_supported(D, feat_dtype))
        return fail(QR_ERR_UNSUPPORTED, "qr_dense_forward_tc: shapes of the tcgen05 path only (D %% 32 == 0, or D < 32 with D %% 4 == 0; D = %d): "
                                        "use qr_dense_forward", D);
    if (!tile_range || !out_map || !final_T || !mean2d || !conic_opac || !features || !ws)
        return fail(QR_ERR_NULL_POINTER, "qr_dense_forward_tc: NULL argument");
    if (!aligned16(out_map) || !aligned16(features) || !aligned16(conic_opac) || !aligned16(mean2d) || !aligned16(ws))
        return fail(QR_ERR_MISALIGNED, "qr_dense_forward_tc: 16-byte alignment");
    const Cam c = make_cam(cam);
    const WsLayout L = ws_layout(c, cap);
    if (ws_bytes < L.total) return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_dense_forward_tc: workspace %zu < %zu bytes", ws_bytes, L.total);
    cudaStream_t st = (cudaStream_t)stream;
    WalkParams2 w2;
    w2.cam = c; w2.K = cap;
    w2.mean2d = reinterpret_cast<const float2*>(mean2d);
    w2.conic_opac = reinterpret_cast<const float4*>(conic_opac);
    w2.isect = isect_gauss; w2.tile_range = reinterpret_cast<const int2*>(tile_range);
    w2.n_sel = nullptr; w2.resid = final_T; w2.sel_idx = nullptr; w2.sel_w = nullptr;
    w2.sl = sel_view(L.sel, ws);
    w2.t_min = t_min;
    if (int rc = launch_walk2_dense(w2, st)) return rc;
    BlendParams bp;
    bp.cam = c; bp.K = cap; bp.D = D; bp.cap = 0; bp.num_tiles = c.tiles_x * c.tiles_y; bp.tile_ticket = nullptr;
    bp.features = features; bp.gcount = nullptr; bp.ucount = nullptr; bp.rec = nullptr;
    bp.n_sel = nullptr; bp.resid = nullptr; bp.out_map = out_map; bp.sel_idx = nullptr; bp.sel_w = nullptr;
    bp.sl = w2.sl;
    bp.feat_f16 = feat_dtype == QR_F16 ? 1 : 0;
    if (int rc = launch_blend_mma(bp, st)) return rc;
    // half tiles whose lists were too small (flag in their header): the FFMA kernel, after the blend has written zeros there
    RenderParams p;
    p.cam = c; p.D = D; p.t_min = t_min;
    p.mean2d = w2.mean2d; p.conic_opac = w2.conic_opac;
    p.isect = isect_gauss; p.tile_range = w2.tile_range; p.features = features;
    p.out_map = out_map; p.final_T = final_T;
    p.only_hdr = w2.sl.hdr;
    return launch_render(p, feat_dtype, st);
}

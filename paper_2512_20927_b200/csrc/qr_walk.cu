// qr_walk.cu -- the O(N) part of qr_forward: Algorithm 1 lines 3-19 for every pixel.
//
// walk2_kernel: CTA = one 16x8-pixel half tile (4 warps), thread = pixel, warp = a WX x (32 / WX) block of pixels.
// The tile's depth-sorted list is staged 128 entries at a time in shared memory.  Per 32 staged entries a warp first
// runs, with lane = entry, an exact conservative test "can the Gaussian's included region (rule R4: power >= -4.5 and
// alpha' >= 1/255) reach any pixel centre of my block" -- the minimum of the conic's quadratic form over the block's
// rectangle against a per-Gaussian bound -- and then, with lane = pixel, walks only the surviving entries, strictly in
// list order, in the fp32 decision arithmetic of DESIGN.md (T is carried sequentially per pixel: no scan, no
// reordering).  The inner step is branch free: a pixel that the Gaussian does not reach, or that has already stopped,
// takes alpha' = 0, which leaves T, k and every comparison of the listing unchanged.
//
// A selection (line 6) is not blended here.  The warp appends one 8-byte entry {w^Q, column | slot | pixel} to its own
// list (no atomics: a list has one writer) and the pixel's Gaussian id to sel_idx; the column is the Gaussian's number
// in the half tile's union of selected Gaussians, handed out on first selection (one shared-memory CAS by lane 0).
// When its pixels have all stopped (T_test < 1/(K+1), lines 15-17) the warp normalises its entries by 1/(1 - T^Q)
// (line 20) in place and scatters them to sel_w.  qr_sel.cuh describes the lists; the forward blend and the backward
// scatter both consume them as they are.
#include "qr_sel.cuh"
#include <stdlib.h>

namespace qr {

constexpr int kW2Threads = 128;
constexpr int kW2Batch = 128;
#ifndef QR_WX
#define QR_WX 16
#endif

__device__ __forceinline__ float clampf(float v, float lo, float hi) { return fminf(fmaxf(v, lo), hi); }
__device__ __forceinline__ void st_release(int32_t* p, int32_t v)
{
    asm volatile("st.release.gpu.global.b32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// min over the rectangle [X0, X1] x [Y0, Y1] of  Q(d) = a dx^2 + 2 b dx dy + c dy^2,  d = point - mean  (power = -Q/2),
// compared with qmax.  Q is convex: if the mean is inside the rectangle the minimum is 0, otherwise it lies on one of
// the four edges, where Q is a 1-D parabola clamped to the edge.  NaNs answer "hit" (conservative).
__device__ __forceinline__ bool rect_hit(float mx, float my, float a, float b, float c, float ia, float ic, float qmax,
                                         float X0, float X1, float Y0, float Y1)
{
    const float dx0 = X0 - mx, dx1 = X1 - mx, dy0 = Y0 - my, dy1 = Y1 - my;
    const bool in = dx0 <= 0.0f && dx1 >= 0.0f && dy0 <= 0.0f && dy1 >= 0.0f;
    const float b2 = b + b;
    float t, q, qmin;
    t = clampf(-b * dy0 * ia, dx0, dx1); qmin = __fmaf_rn(__fmaf_rn(a, t, b2 * dy0), t, c * dy0 * dy0);
    t = clampf(-b * dy1 * ia, dx0, dx1); q = __fmaf_rn(__fmaf_rn(a, t, b2 * dy1), t, c * dy1 * dy1); qmin = fminf(qmin, q);
    t = clampf(-b * dx0 * ic, dy0, dy1); q = __fmaf_rn(__fmaf_rn(c, t, b2 * dx0), t, a * dx0 * dx0); qmin = fminf(qmin, q);
    t = clampf(-b * dx1 * ic, dy0, dy1); q = __fmaf_rn(__fmaf_rn(c, t, b2 * dx1), t, a * dx1 * dx1); qmin = fminf(qmin, q);
    if (in) qmin = 0.0f;
    return !(qmin > qmax);
}

// MODE 0: Q-Render (Algorithm 1).  MODE 1: stratified-K pass 2 (reading R18): the same walk with
// the per-pixel boundaries b_k = clamp(mu + sigma z_k, 0, 1) in place of 1 - (k+1)/(K+1).  MODE 2: stratified-K pass 1: the
// dense transmittance statistics (mu, sigma) of every pixel, nothing else.
// MODE 3: DENSE (the comparator, Eq. 1 / qr_dense_forward on the tensor cores): every blended entry is emitted with its dense weight
// T alpha' (stop rule R7 at t_min, no normalisation, no records); the lists have the capacity of K = p.K entries per pixel on
// average, a half tile that needs more is flagged (hdr[5] = 1, empty lists) and left to the FFMA kernel.
enum { kWalkQ = 0, kWalkStrat = 1, kWalkStats = 2, kWalkDense = 3 };

template <int WX, int MODE>
__global__ void __launch_bounds__(kW2Threads, 10) walk2_kernel(const WalkParams2 p)
{
    constexpr int WY = 32 / WX;
    __shared__ float4 s_co[kW2Batch];      // a, b, c, opacity
    __shared__ float4 s_cull[kW2Batch];    // 1/a, 1/c, qmax, -
    __shared__ float2 s_xy[kW2Batch];
    __shared__ int32_t s_id[kW2Batch];
    __shared__ int32_t s_col[kW2Batch];    // column of a staged entry in the union, -1 = not selected yet, -2 = being numbered
    __shared__ float thr[QR_MAX_K + 1];
    __shared__ float zs[MODE == kWalkStrat ? QR_MAX_K + 1 : 1];     // z_k of the stratified boundaries
    __shared__ int32_t s_ucount, s_evals, s_consumed, s_ovf;

    __shared__ int32_t s_ht;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int K = p.K;
    const int num_half = p.cam.tiles_x * p.cam.tiles_y * 2;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const uint32_t s_col_addr = (uint32_t)__cvta_generic_to_shared(s_col);
    const uint32_t s_ucount_addr = (uint32_t)__cvta_generic_to_shared(&s_ucount);
    const uint32_t s_co_addr = (uint32_t)__cvta_generic_to_shared(s_co);
    const uint32_t s_xy_addr = (uint32_t)__cvta_generic_to_shared(s_xy);
    const uint32_t s_id_addr = (uint32_t)__cvta_generic_to_shared(s_id);
    const uint32_t thr_addr = (uint32_t)__cvta_generic_to_shared(thr);
    for (int k = tid; k <= K; k += kW2Threads)                            // thresholds as printed (R3)
        thr[k] = __fsub_rn(1.0f, __fdiv_rn((float)(k + 1), (float)(K + 1)));
    if (MODE == kWalkStrat)
        for (int k = tid; k <= K; k += kW2Threads)
            zs[k] = __fmul_rn(p.z_max, __fsub_rn(1.0f, __fdiv_rn((float)(2 * (k + 1)), (float)(K + 1))));
    const float t_break_q = __fdiv_rn(1.0f, (float)(K + 1));
    // the blend kernel (launched with programmatic stream serialization) may start as soon as every walk CTA is resident:
    // it consumes half tiles as their flags are released and shares the SMs with this kernel
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (tid == 0) stamp_time(p.sl.ctrl, 0, true);
    if (MODE != kWalkStats && blockIdx.x == 0 && tid == 0) {
        p.sl.stamp[0] = kSelMagic; p.sl.stamp[1] = p.cam.width; p.sl.stamp[2] = p.cam.height; p.sl.stamp[3] = K;
        const unsigned long long a = (unsigned long long)p.sel_idx;
        p.sl.stamp[4] = (int32_t)(a & 0xffffffffull); p.sl.stamp[5] = (int32_t)(a >> 32);
    }

  // Persistent CTAs: half tiles are handed out in index order by a global ticket (the blend kernel, which may already be
  // running, consumes them in the same order); when a half tile's lists are complete its ready flag is released.
  int prev_ht = -1;
  long long prev_start = 0;
  while (true) {
    __syncthreads();                                   // everybody is through with the previous half tile: its lists are written
    if (tid == 0) {
        // publish the previous half tile.  One release per CTA: the block barrier orders every thread's list, record and
        // header stores before this thread's st.release, which is cumulative (no per-warp __threadfence: with the blend
        // streaming the map through the same memory system a fence costs microseconds)
        if (MODE != kWalkStats && prev_ht >= 0) {
            int32_t* h = p.sl.hdr + (size_t)prev_ht * kHdrWords;
            h[4] = s_ucount; h[5] = 0; h[6] = s_consumed; h[7] = s_evals; h[8] = (int32_t)(clock64() - prev_start);
            if (MODE == kWalkDense && s_ovf) { h[0] = h[1] = h[2] = h[3] = 0; h[4] = 0; h[5] = 1; }      // lists too small: FFMA kernel
            st_release(p.sl.flags + prev_ht, 1);
        }
        s_ht = atomicAdd(p.sl.ctrl, 1); s_ucount = 0; s_evals = 0; s_consumed = 0; s_ovf = 0;
    }
    __syncthreads();
    const int ht = s_ht;
    if (ht >= num_half) { if (tid == 0) stamp_time(p.sl.ctrl, 1, false); break; }
    prev_ht = -1;
    const int tile = ht >> 1;
    const int x0 = (tile % p.cam.tiles_x) * kTile, y0 = (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8;
    int32_t* hdr = p.sl.hdr + (size_t)ht * kHdrWords;
    if (y0 >= p.cam.height) {                         // half tile below the image: empty lists
        if (MODE != kWalkStats) {
            if (tid < kHdrWords) { hdr[tid] = 0; __threadfence(); }
            __syncthreads();
            if (tid == 0) { __threadfence(); st_release(p.sl.flags + ht, 1); }
        }
        continue;
    }
    // block of this warp and pixel of this lane
    const int bx0 = WX == 16 ? 0 : 8 * (warp & 1), by0 = WX == 16 ? 2 * warp : 4 * (warp >> 1);
    const int lx = lane & (WX - 1), ly = lane / WX;
    const int mpix = (by0 + ly) * kTile + bx0 + lx;   // row-major index inside the half tile
    const int px = x0 + bx0 + lx, py = y0 + by0 + ly;
    const bool inside = px < p.cam.width && py < p.cam.height;
    // batch of views stacked as one tall tile grid (qr_forward_batch): alpha' is evaluated in the view's own pixel
    // coordinates, exactly as a single-view call would; only the output index uses the tall row
    const int yoff = p.view_h > 0 ? (y0 / p.view_h) * p.view_h : 0;
    const float fpx = (float)px + 0.5f, fpy = (float)(py - yoff) + 0.5f;          // R5
    const float X0 = (float)(x0 + bx0) + 0.5f, X1 = X0 + (float)(WX - 1);
    const float Y0 = (float)(y0 - yoff + by0) + 0.5f, Y1 = Y0 + (float)(WY - 1);
    const int64_t pix = (int64_t)py * p.cam.width + px;
    int32_t* my_idx = p.sel_idx + pix * K;
    uint2* my_ent = p.sl.ent + ((size_t)ht * kSelLists + warp) * p.sl.qcap;
    int32_t* uid_g = p.sl.uid + (size_t)ht * p.sl.ucap;
    const long long t_start = clock64();
    const int2 range = p.tile_range[tile];

    bool done = !inside;
    float T = 1.0f, TQ = 1.0f;
    // boundary k of this pixel: Algorithm 1's 1 - (k+1)/(K+1), or the stratified one (sigma == 0: the uniform one)
    float mu = 0.0f, sg = 0.0f;
    if (MODE == kWalkStrat && inside) { const float2 st = p.stats[pix]; mu = st.x; sg = st.y; }
    auto bnd = [&](int kk) -> float {
        float u;
        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(u) : "r"(thr_addr + 4u * (uint32_t)kk));
        if (MODE == kWalkStrat) {
            const float b = fminf(fmaxf(__fmaf_rn(sg, zs[kk], mu), 0.0f), 1.0f);
            if (sg > 0.0f) u = kk >= K ? 0.0f : b;
        }
        return u;
    };
    float thr_k = bnd(0);
    const float t_break = MODE == kWalkQ ? t_break_q : (MODE == kWalkStrat ? fmaxf(bnd(K - 1), p.t_min) : p.t_min);
    float S1 = 0.0f, S2 = 0.0f;                 // MODE 2: sums of T and T^2 over the entries that get a dense weight
    int nd = 0;
    int k = 0, ns = 0, n_ent = 0, n_eval = 0, consumed = 0;
    int32_t* idx_ptr = my_idx;                  // next slot of this pixel's selection record
    uint2* ent_ptr = my_ent;                    // end of this warp's entry list (warp-uniform)
    uint32_t slotpix = (uint32_t)mpix;          // slot << 7 | pixel of this pixel's next entry
    bool warp_done = __all_sync(0xffffffffu, done);

    // alpha' of staged entry e at this pixel (Eq. 1) with inclusion rule R4, fp32 decision arithmetic;
    // 0 = the Gaussian is not in I for this pixel
    auto alpha_of = [&](int e) -> float {
        float4 co; float2 xy;
        asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(co.x), "=f"(co.y), "=f"(co.z), "=f"(co.w) : "r"(s_co_addr + 16u * (uint32_t)e));
        asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(xy.x), "=f"(xy.y) : "r"(s_xy_addr + 8u * (uint32_t)e));
        const float dx = __fsub_rn(fpx, xy.x), dy = __fsub_rn(fpy, xy.y);
        const float q1 = __fmul_rn(__fmul_rn(co.x, dx), dx);
        const float q2 = __fmaf_rn(__fmul_rn(co.z, dy), dy, q1);
        const float q3 = __fmul_rn(__fmul_rn(co.y, dx), dy);
        const float power = __fmaf_rn(-0.5f, q2, -q3);
        float a = fminf(kAlphaMax, __fmul_rn(co.w, expf(power)));
        if (power > 0.0f || power < kPowerMin || a < kAlphaMin) a = 0.0f;
        return a;
    };
    // Algorithm 1 lines 5-18 for staged entry e with this pixel's alpha' = a (0: a no-op, T_test = T)
    auto step = [&](int e, float a) {
        if (done) a = 0.0f;
        const float oma = __fsub_rn(1.0f, a);
        const float T_test = __fmul_rn(T, oma);                                  // line 5
        if (MODE == kWalkStats) {               // pass 1 of stratified-K: T_i of every entry before the dense stop R7
            if (a > 0.0f) {
                if (T_test < t_break) done = true;
                else { T = T_test; S1 = __fadd_rn(S1, T); S2 = __fmaf_rn(T, T, S2); ++nd; }
            }
            return;
        }
        bool sel;
        if (MODE == kWalkDense) {                                                // R7: stop before blending the entry that takes T below t_min
            const bool stop = a > 0.0f && T_test < t_break;
            sel = a > 0.0f && !stop;
            if (stop) done = true;
        } else sel = T_test < thr_k;                                             // line 6
        const uint32_t sm = __ballot_sync(0xffffffffu, sel);
        if (sm) {
            // column of this Gaussian in the half tile's union: the first warp to select it numbers it
            int col = 0;
            int32_t id;
            asm volatile("ld.shared.b32 %0, [%1];" : "=r"(id) : "r"(s_id_addr + 4u * (uint32_t)e));
            if (lane == 0) {
                const uint32_t slot = s_col_addr + 4u * (uint32_t)e;
                int old;
                asm volatile("atom.shared.cas.b32 %0, [%1], -1, -2;" : "=r"(old) : "r"(slot) : "memory");
                if (old == -1) {
                    asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(col) : "r"(s_ucount_addr) : "memory");
                    if (MODE != kWalkDense || col < p.sl.ucap) uid_g[col] = id;
                    asm volatile("st.volatile.shared.b32 [%0], %1;" ::"r"(slot), "r"(col) : "memory");
                } else {
                    col = old;
                    while (col == -2) asm volatile("ld.volatile.shared.b32 %0, [%1];" : "=r"(col) : "r"(slot) : "memory");
                }
            }
            col = __shfl_sync(0xffffffffu, col, 0);
            if (MODE == kWalkDense) {
                const int ne = __popc(sm);
                if (n_ent + ne <= p.sl.qcap && col < p.sl.ucap) {                // warp-uniform
                    if (sel) ent_ptr[__popc(sm & lt_mask)] = make_uint2(__float_as_uint(__fmul_rn(T, a)), ((uint32_t)col << 15) | (uint32_t)mpix);
                    ent_ptr += ne;
                    n_ent += ne;
                } else if (lane == 0) s_ovf = 1;
                if (sel) T = T_test;
                return;
            }
            if (sel) {
                const float wQ = __fmul_rn(TQ, a);                               // line 8
                *idx_ptr++ = id;
                ent_ptr[__popc(sm & lt_mask)] = make_uint2(__float_as_uint(wQ), ((uint32_t)col << 15) | slotpix);
                slotpix += 128u;                                                 // next slot of this pixel
                ++ns;                                                            // line 9 runs in the blend
                k = k + 1;                                                       // line 7
                TQ = __fmul_rn(TQ, oma);                                         // line 10
                float tk;
                while (true) {                                                   // lines 11-13
                    tk = bnd(k);
                    if (!(T_test < tk)) break;
                    k = k + 1;
                }
                thr_k = tk;
            }
            const int ne = __popc(sm);
            ent_ptr += ne;
            n_ent += ne;
        }
        if (MODE == kWalkDense) return;                                          // (nothing selected in the warp: sel is false here)
        if (T_test < t_break) done = true;                                       // lines 15-17
        else T = T_test;                                                         // line 18
    };

    for (int b0 = range.x; b0 < range.y; b0 += kW2Batch) {
        if (__syncthreads_and(warp_done)) break;                          // every pixel of the half tile has stopped
        {   // ---- stage the batch ----
            const int idx = b0 + tid;
            int32_t id = -1;
            float4 co = make_float4(1.f, 0.f, 1.f, 0.f), cull = make_float4(1.f, 1.f, -1.f, 0.f);   // never hit
            float2 xy = make_float2(0.f, 0.f);
            if (idx < range.y) {
                id = (int32_t)p.isect[idx];
                xy = __ldg(p.mean2d + id);
                co = __ldg(p.conic_opac + id);
                // included  =>  Q <= 9 (power >= -4.5)  and  opacity exp(-Q/2) >= 1/255  <=>  Q <= 2 ln(255 opacity).
                // 1e-4 relative + 1e-3 absolute slack covers the different rounding of Q here and of `power` below.
                float qmax = fminf(9.0f, 2.0f * __logf(255.0f * co.w)) * 1.0001f + 1e-3f;
                const bool valid = co.x > 0.0f && co.z > 0.0f && co.x * co.z - co.y * co.y > 0.0f;
                float ia = 0.0f, ic = 0.0f;
                if (valid) { ia = 1.0f / co.x; ic = 1.0f / co.z; }
                else qmax = 3.0e38f;                                      // odd conic: never culled
                if (!(co.w > 0.0f)) qmax = -1.0f;                         // alpha' = 0 < 1/255 everywhere
                cull = make_float4(ia, ic, qmax, 0.f);
            }
            if (p.batch_n > 0 && id >= 0) id = (int32_t)((uint32_t)id % (uint32_t)p.batch_n);     // virtual Gaussian b N + i -> i
            s_id[tid] = id; s_co[tid] = co; s_xy[tid] = xy; s_cull[tid] = cull; s_col[tid] = -1;
        }
        __syncthreads();
        if (warp_done) continue;
        const int nb = min(kW2Batch, range.y - b0);
        consumed = b0 + nb - range.x;

        for (int c = 0; c < nb; c += 32) {
            uint32_t m;
            {   // lane = entry: which of these 32 Gaussians can reach a pixel centre of my block
                const float4 co = s_co[c + lane], cu = s_cull[c + lane];
                const float2 xy = s_xy[c + lane];
                m = __ballot_sync(0xffffffffu, rect_hit(xy.x, xy.y, co.x, co.y, co.z, cu.x, cu.y, cu.z, X0, X1, Y0, Y1));
            }
            n_eval += __popc(m);
            // lane = pixel.  Two surviving entries per iteration: their alpha' evaluations are independent and
            // interleave; the transmittance steps (lines 5-18) then run one after the other, in list order.
            while (m) {
                const int e0 = c + __ffs(m) - 1;
                m &= m - 1;
                const bool two = m != 0;
                const int e1 = two ? c + __ffs(m) - 1 : e0;
                m &= m - 1;
                float a0 = alpha_of(e0), a1 = alpha_of(e1);
                if (!two) a1 = 0.0f;
                step(e0, a0);
                step(e1, a1);
            }
            if (__all_sync(0xffffffffu, done)) { warp_done = true; break; }
        }
    }

    // ---- the warp's pixels: n_sel, T^Q; its entries: x 1/(1 - T^Q) (line 20), scattered to sel_w ----
    if (MODE == kWalkStats) {
        if (inside) {
            float m = 0.0f, sd = 0.0f;
            if (nd > 0) {
                m = __fdiv_rn(S1, (float)nd);
                const float var = __fsub_rn(__fdiv_rn(S2, (float)nd), __fmul_rn(m, m));
                sd = __fsqrt_rn(fmaxf(var, 0.0f));
            }
            p.stats[pix] = make_float2(m, sd);
        }
        continue;
    }
    if (MODE == kWalkDense) {                  // weights are final (Eq. 1 is not normalised); final_T = T
        if (inside) p.resid[pix] = T;
        if (lane == 0) {
            hdr[warp] = n_ent;
            atomicAdd(&s_evals, n_eval);
            atomicMax(&s_consumed, consumed);
        }
        prev_ht = ht; prev_start = t_start;
        continue;
    }
    const float inv = ns > 0 ? __fdiv_rn(1.0f, __fsub_rn(1.0f, TQ)) : 0.0f;
    if (inside) {
        p.n_sel[pix] = ns;
        p.resid[pix] = ns > 0 ? TQ : 1.0f;                                               // R8
    }
    __syncwarp();
    constexpr int kPre = 8;                     // entries a lane re-reads at once: the L2 round trips overlap
    for (int i0 = 0; i0 < n_ent; i0 += 32 * kPre) {
        uint2 en[kPre];
#pragma unroll
        for (int u = 0; u < kPre; ++u) {
            const int i = i0 + u * 32 + lane;
            en[u] = i < n_ent ? __ldcg(my_ent + i) : make_uint2(0u, 0u);
        }
#pragma unroll
        for (int u = 0; u < kPre; ++u) {
            const int i = i0 + u * 32 + lane;
            const int pm = sel_pixel(en[u].y);
            const int src = WX == 16 ? (pm & 31) : (((pm >> 4) & 3) * 8 + (pm & 7));     // lane that owns pixel pm
            const float inv_p = __shfl_sync(0xffffffffu, inv, src);
            if (i < n_ent) {
                const float w = __fmul_rn(__uint_as_float(en[u].x), inv_p);
                my_ent[i].x = __float_as_uint(w);
                const int64_t q = (int64_t)(y0 + (pm >> 4)) * p.cam.width + x0 + (pm & 15);
                p.sel_w[q * K + sel_slot(en[u].y)] = w;
            }
        }
    }
    if (lane == 0) {
        hdr[warp] = n_ent;
        atomicAdd(&s_evals, n_eval);
        atomicMax(&s_consumed, consumed);
    }
    prev_ht = ht; prev_start = t_start;                        // published by thread 0 after the barrier at the loop top
  }
}

// ------------------------------------------------------------------------------------------------------------------
// walk2_multi_kernel: Algorithm 1 for NK values of K in ONE pass over the lists ("multi-K in one walk").
// What the K share: the staged batch, the culling test, alpha' and the dense transmittance T (line 5 / line 18 do not depend
// on K).  What each K keeps: its boundaries 1 - (k+1)/(K+1), its index k, T^Q, its stop test T_test < 1/(K+1), its records and
// its selection lists with their own union numbering (the workspaces are qr_forward's, one per K, so qr_backward_lists and
// the blend take them as they are).  For every K the decisions and the fp32 values are those of walk2_kernel run with that K:
// T evolves identically while the K is active, and a K that has stopped for a pixel selects nothing more there.
// ------------------------------------------------------------------------------------------------------------------
template <int NK>
__global__ void __launch_bounds__(kW2Threads, 4) walk2_multi_kernel(const WalkParamsMulti p)
{
    constexpr int WX = 16, WY = 2;
    __shared__ float4 s_co[kW2Batch];
    __shared__ float4 s_cull[kW2Batch];
    __shared__ float2 s_xy[kW2Batch];
    __shared__ int32_t s_id[kW2Batch];
    __shared__ int32_t s_col[NK][kW2Batch];
    __shared__ float thr[NK][QR_MAX_K + 1];
    __shared__ int32_t s_ucount[NK], s_evals, s_consumed, s_ht;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int num_half = p.cam.tiles_x * p.cam.tiles_y * 2;
    const uint32_t lt_mask = (1u << lane) - 1u;
    int Kj[NK];
    float t_break[NK];
#pragma unroll
    for (int j = 0; j < NK; ++j) {
        Kj[j] = p.K[j];
        for (int k = tid; k <= Kj[j]; k += kW2Threads)                    // thresholds as printed (R3)
            thr[j][k] = __fsub_rn(1.0f, __fdiv_rn((float)(k + 1), (float)(Kj[j] + 1)));
        t_break[j] = __fdiv_rn(1.0f, (float)(Kj[j] + 1));
    }
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (blockIdx.x == 0 && tid == 0) {
#pragma unroll
        for (int j = 0; j < NK; ++j) {
            int32_t* sp = p.sl[j].stamp;
            sp[0] = kSelMagic; sp[1] = p.cam.width; sp[2] = p.cam.height; sp[3] = Kj[j];
            const unsigned long long a = (unsigned long long)p.sel_idx[j];
            sp[4] = (int32_t)(a & 0xffffffffull); sp[5] = (int32_t)(a >> 32);
            stamp_time(p.sl[j].ctrl, 0, true);
        }
    }

  int prev_ht = -1;
  long long prev_start = 0;
  while (true) {
    __syncthreads();
    if (tid == 0) {
        if (prev_ht >= 0) {
#pragma unroll
            for (int j = 0; j < NK; ++j) {
                int32_t* h = p.sl[j].hdr + (size_t)prev_ht * kHdrWords;
                h[4] = s_ucount[j]; h[5] = 0; h[6] = s_consumed; h[7] = s_evals; h[8] = (int32_t)(clock64() - prev_start);
                st_release(p.sl[j].flags + prev_ht, 1);
            }
        }
        s_ht = atomicAdd(p.sl[0].ctrl, 1); s_evals = 0; s_consumed = 0;
#pragma unroll
        for (int j = 0; j < NK; ++j) s_ucount[j] = 0;
    }
    __syncthreads();
    const int ht = s_ht;
    if (ht >= num_half) {
        if (tid == 0)
            for (int j = 0; j < NK; ++j) stamp_time(p.sl[j].ctrl, 1, false);
        break;
    }
    prev_ht = -1;
    const int tile = ht >> 1;
    const int x0 = (tile % p.cam.tiles_x) * kTile, y0 = (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8;
    if (y0 >= p.cam.height) {                         // half tile below the image: empty lists
#pragma unroll
        for (int j = 0; j < NK; ++j)
            if (tid < kHdrWords) p.sl[j].hdr[(size_t)ht * kHdrWords + tid] = 0;
        __threadfence();
        __syncthreads();
        if (tid == 0) {
            __threadfence();
            for (int j = 0; j < NK; ++j) st_release(p.sl[j].flags + ht, 1);
        }
        continue;
    }
    const int by0 = 2 * warp;
    const int lx = lane & (WX - 1), ly = lane / WX;
    const int mpix = (by0 + ly) * kTile + lx;
    const int px = x0 + lx, py = y0 + by0 + ly;
    const bool inside = px < p.cam.width && py < p.cam.height;
    const float fpx = (float)px + 0.5f, fpy = (float)py + 0.5f;          // R5
    const float X0 = (float)x0 + 0.5f, X1 = X0 + (float)(WX - 1);
    const float Y0 = (float)(y0 + by0) + 0.5f, Y1 = Y0 + (float)(WY - 1);
    const int64_t pix = (int64_t)py * p.cam.width + px;
    const long long t_start = clock64();
    const int2 range = p.tile_range[tile];

    // per-K state of this pixel / this warp
    int32_t* idx_ptr[NK]; uint2* my_ent[NK]; uint2* ent_ptr[NK]; int32_t* uid_g[NK];
    float thr_k[NK], TQ[NK];
    int k[NK], ns[NK], n_ent[NK];
    uint32_t slotpix[NK];
    bool dn[NK];
#pragma unroll
    for (int j = 0; j < NK; ++j) {
        idx_ptr[j] = p.sel_idx[j] + pix * Kj[j];
        my_ent[j] = p.sl[j].ent + ((size_t)ht * kSelLists + warp) * p.sl[j].qcap;
        ent_ptr[j] = my_ent[j];
        uid_g[j] = p.sl[j].uid + (size_t)ht * p.sl[j].ucap;
        thr_k[j] = thr[j][0]; TQ[j] = 1.0f; k[j] = 0; ns[j] = 0; n_ent[j] = 0; slotpix[j] = (uint32_t)mpix; dn[j] = !inside;
    }
    bool done = !inside;                        // every K has stopped for this pixel
    float T = 1.0f;
    int n_eval = 0, consumed = 0;
    bool warp_done = __all_sync(0xffffffffu, done);

    // alpha' of staged entry e at this pixel (Eq. 1) with inclusion rule R4, fp32 decision arithmetic
    auto alpha_of = [&](int e) -> float {
        const float4 co = s_co[e];
        const float2 xy = s_xy[e];
        const float dx = __fsub_rn(fpx, xy.x), dy = __fsub_rn(fpy, xy.y);
        const float q1 = __fmul_rn(__fmul_rn(co.x, dx), dx);
        const float q2 = __fmaf_rn(__fmul_rn(co.z, dy), dy, q1);
        const float q3 = __fmul_rn(__fmul_rn(co.y, dx), dy);
        const float power = __fmaf_rn(-0.5f, q2, -q3);
        float a = fminf(kAlphaMax, __fmul_rn(co.w, expf(power)));
        if (power > 0.0f || power < kPowerMin || a < kAlphaMin) a = 0.0f;
        return a;
    };
    // Algorithm 1 lines 5-18 for staged entry e, once for the shared T and once per K for the selection
    auto step = [&](int e, float a) {
        if (done) a = 0.0f;
        const float oma = __fsub_rn(1.0f, a);
        const float T_test = __fmul_rn(T, oma);                                  // line 5
        const int32_t id = s_id[e];
        bool all = true;
#pragma unroll
        for (int j = 0; j < NK; ++j) {
            const bool sel = !dn[j] && T_test < thr_k[j];                        // line 6
            const uint32_t sm = __ballot_sync(0xffffffffu, sel);
            if (sm) {
                int col = 0;
                if (lane == 0) {
                    const uint32_t slot = (uint32_t)__cvta_generic_to_shared(&s_col[j][e]);
                    int old;
                    asm volatile("atom.shared.cas.b32 %0, [%1], -1, -2;" : "=r"(old) : "r"(slot) : "memory");
                    if (old == -1) {
                        col = atomicAdd(&s_ucount[j], 1);
                        uid_g[j][col] = id;
                        asm volatile("st.volatile.shared.b32 [%0], %1;" ::"r"(slot), "r"(col) : "memory");
                    } else {
                        col = old;
                        while (col == -2) asm volatile("ld.volatile.shared.b32 %0, [%1];" : "=r"(col) : "r"(slot) : "memory");
                    }
                }
                col = __shfl_sync(0xffffffffu, col, 0);
                if (sel) {
                    const float wQ = __fmul_rn(TQ[j], a);                        // line 8
                    *idx_ptr[j]++ = id;
                    ent_ptr[j][__popc(sm & lt_mask)] = make_uint2(__float_as_uint(wQ), ((uint32_t)col << 15) | slotpix[j]);
                    slotpix[j] += 128u;
                    ++ns[j];
                    k[j] = k[j] + 1;                                             // line 7
                    TQ[j] = __fmul_rn(TQ[j], oma);                               // line 10
                    float tk;
                    while (true) {                                               // lines 11-13
                        tk = thr[j][k[j]];
                        if (!(T_test < tk)) break;
                        k[j] = k[j] + 1;
                    }
                    thr_k[j] = tk;
                }
                const int ne = __popc(sm);
                ent_ptr[j] += ne;
                n_ent[j] += ne;
            }
            if (!dn[j] && T_test < t_break[j]) dn[j] = true;                     // lines 15-17 for this K
            all = all && dn[j];
        }
        if (all) done = true;
        else T = T_test;                                                         // line 18
    };

    for (int b0 = range.x; b0 < range.y; b0 += kW2Batch) {
        if (__syncthreads_and(warp_done)) break;                          // every pixel of the half tile has stopped for every K
        {   // ---- stage the batch (as walk2_kernel) ----
            const int idx = b0 + tid;
            int32_t id = -1;
            float4 co = make_float4(1.f, 0.f, 1.f, 0.f), cull = make_float4(1.f, 1.f, -1.f, 0.f);   // never hit
            float2 xy = make_float2(0.f, 0.f);
            if (idx < range.y) {
                id = (int32_t)p.isect[idx];
                xy = __ldg(p.mean2d + id);
                co = __ldg(p.conic_opac + id);
                float qmax = fminf(9.0f, 2.0f * __logf(255.0f * co.w)) * 1.0001f + 1e-3f;
                const bool valid = co.x > 0.0f && co.z > 0.0f && co.x * co.z - co.y * co.y > 0.0f;
                float ia = 0.0f, ic = 0.0f;
                if (valid) { ia = 1.0f / co.x; ic = 1.0f / co.z; }
                else qmax = 3.0e38f;
                if (!(co.w > 0.0f)) qmax = -1.0f;
                cull = make_float4(ia, ic, qmax, 0.f);
            }
            s_id[tid] = id; s_co[tid] = co; s_xy[tid] = xy; s_cull[tid] = cull;
#pragma unroll
            for (int j = 0; j < NK; ++j) s_col[j][tid] = -1;
        }
        __syncthreads();
        if (warp_done) continue;
        const int nb = min(kW2Batch, range.y - b0);
        consumed = b0 + nb - range.x;
        for (int c = 0; c < nb; c += 32) {
            uint32_t m;
            {
                const float4 co = s_co[c + lane], cu = s_cull[c + lane];
                const float2 xy = s_xy[c + lane];
                m = __ballot_sync(0xffffffffu, rect_hit(xy.x, xy.y, co.x, co.y, co.z, cu.x, cu.y, cu.z, X0, X1, Y0, Y1));
            }
            n_eval += __popc(m);
            while (m) {
                const int e0 = c + __ffs(m) - 1;
                m &= m - 1;
                const bool two = m != 0;
                const int e1 = two ? c + __ffs(m) - 1 : e0;
                m &= m - 1;
                float a0 = alpha_of(e0), a1 = alpha_of(e1);
                if (!two) a1 = 0.0f;
                step(e0, a0);
                step(e1, a1);
            }
            if (__all_sync(0xffffffffu, done)) { warp_done = true; break; }
        }
    }

    // ---- per K: n_sel, T^Q; the warp's entries x 1/(1 - T^Q) (line 20), scattered to sel_w ----
    int32_t* hdr0 = nullptr;
#pragma unroll
    for (int j = 0; j < NK; ++j) {
        const int K = Kj[j];
        const float inv = ns[j] > 0 ? __fdiv_rn(1.0f, __fsub_rn(1.0f, TQ[j])) : 0.0f;
        if (inside) {
            p.n_sel[j][pix] = ns[j];
            p.resid[j][pix] = ns[j] > 0 ? TQ[j] : 1.0f;                                  // R8
        }
        __syncwarp();
        constexpr int kPre = 8;
        for (int i0 = 0; i0 < n_ent[j]; i0 += 32 * kPre) {
            uint2 en[kPre];
#pragma unroll
            for (int u = 0; u < kPre; ++u) {
                const int i = i0 + u * 32 + lane;
                en[u] = i < n_ent[j] ? __ldcg(my_ent[j] + i) : make_uint2(0u, 0u);
            }
#pragma unroll
            for (int u = 0; u < kPre; ++u) {
                const int i = i0 + u * 32 + lane;
                const int pm = sel_pixel(en[u].y);
                const float inv_p = __shfl_sync(0xffffffffu, inv, pm & 31);              // lane that owns pixel pm (WX = 16)
                if (i < n_ent[j]) {
                    const float w = __fmul_rn(__uint_as_float(en[u].x), inv_p);
                    my_ent[j][i].x = __float_as_uint(w);
                    const int64_t q = (int64_t)(y0 + (pm >> 4)) * p.cam.width + x0 + (pm & 15);
                    p.sel_w[j][q * K + sel_slot(en[u].y)] = w;
                }
            }
        }
        if (lane == 0) p.sl[j].hdr[(size_t)ht * kHdrWords + warp] = n_ent[j];
    }
    (void)hdr0;
    if (lane == 0) {
        atomicAdd(&s_evals, n_eval);
        atomicMax(&s_consumed, consumed);
    }
    prev_ht = ht; prev_start = t_start;
  }
}

int launch_walk2_multi(const WalkParamsMulti& p, cudaStream_t st)
{
    const int num_half = p.cam.tiles_x * p.cam.tiles_y * 2;
    for (int j = 0; j < p.nK; ++j)
        QR_CUDA_OK(cudaMemsetAsync(p.sl[j].ctrl, 0, (size_t)(kCtrlWords + num_half) * 4, st));
    const unsigned grid = (unsigned)min(num_half, sm_count() * 4);
    switch (p.nK) {
    case 1:
        QR_CUDA_OK(cudaFuncSetAttribute(walk2_multi_kernel<1>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        walk2_multi_kernel<1><<<grid, kW2Threads, 0, st>>>(p); break;
    case 2:
        QR_CUDA_OK(cudaFuncSetAttribute(walk2_multi_kernel<2>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        walk2_multi_kernel<2><<<grid, kW2Threads, 0, st>>>(p); break;
    case 3:
        QR_CUDA_OK(cudaFuncSetAttribute(walk2_multi_kernel<3>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        walk2_multi_kernel<3><<<grid, kW2Threads, 0, st>>>(p); break;
    default:
        QR_CUDA_OK(cudaFuncSetAttribute(walk2_multi_kernel<4>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        walk2_multi_kernel<4><<<grid, kW2Threads, 0, st>>>(p); break;
    }
    QR_LAUNCH_OK("walk2_multi_kernel");
    return QR_OK;
}

template <int MODE>
static int launch_walk2_mode(const WalkParams2& p, cudaStream_t st)
{
    const int num_half = p.cam.tiles_x * p.cam.tiles_y * 2;
    // tickets and ready flags of this frame
    QR_CUDA_OK(cudaMemsetAsync(p.sl.ctrl, 0, (size_t)(kCtrlWords + num_half) * 4, st));
    const int sms = sm_count();
    const char* e = getenv("QR_WALK_CTAS");           // profiling knob: walk CTAs per SM
    const int per_sm = e ? atoi(e) : 5;
    // the blend kernel takes over the SMs as these CTAs drain (programmatic dependent launch) and needs ~200 KB of shared
    // memory there: an SM only changes its L1 / shared split when it is idle, so this kernel asks for the largest
    // shared-memory carve-out although it uses 8 KB
    QR_CUDA_OK(cudaFuncSetAttribute(walk2_kernel<QR_WX, MODE>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    const unsigned grid = (unsigned)min(num_half, sms * per_sm);
    walk2_kernel<QR_WX, MODE><<<grid, kW2Threads, 0, st>>>(p);
    QR_LAUNCH_OK("walk2_kernel");
    return QR_OK;
}

int launch_walk2(const WalkParams2& p, cudaStream_t st) { return launch_walk2_mode<kWalkQ>(p, st); }
int launch_walk2_dense(const WalkParams2& p, cudaStream_t st) { return launch_walk2_mode<kWalkDense>(p, st); }

// stratified-K: pass 1 (statistics into p.stats), then pass 2 (the walk with the stratified boundaries)
int launch_walk2_stratified(const WalkParams2& p, cudaStream_t st)
{
    if (int rc = launch_walk2_mode<kWalkStats>(p, st)) return rc;
    return launch_walk2_mode<kWalkStrat>(p, st);
}

}  // namespace qr

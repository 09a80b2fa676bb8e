// qr_forward.cu -- qr_forward: Algorithm 1 for every pixel, then f~^Q = f^Q / (1 - T^Q).
//
// The call is split where the method itself splits (the O(N) transmittance walk, the O(KC) blend):
//   D % 32 == 0 or D < 32, D % 4 == 0 (padded to whole 128-channel tiles by TMA)   walk2_kernel (qr_walk.cu: selection lists per 16x8 half tile) -> blend_mma_kernel
//                                 (qr_blend_mma.cu: the blend as a tcgen05 contraction); the dispatcher is at the end of
//                                 this file
//   every other shape             the kernels of THIS file:
// walk_kernel     -- CTA = one 16x16 tile, thread = pixel, warp = 16x2 pixels = four 4x2-pixel groups.  The tile's
//   depth-sorted list is staged 256 entries at a time in shared memory; each warp first intersects the batch with its own
//   pixel rectangle (lane-parallel box test + ballot), then runs Algorithm 1 lines 3-19 sequentially per pixel over the
//   surviving entries only, in the paper's order and in the fp32 decision arithmetic of DESIGN.md.  A selected Gaussian is
//   not blended here: per 4x2 pixel group the kernel appends one record (Gaussian id, the 8 pixels' weights w^Q, 0 where
//   a pixel did not select it) to the group's list in the workspace -- the group's union of selected Gaussians, in depth
//   order.  After the walk the same warp writes n_sel, T^Q and the used slots of the per-pixel selection records
//   sel_idx / sel_w from the group lists it has just written.
// blend_tu_kernel -- D % 4 == 0 outside the tcgen05 shapes (e.g. D = 132): persistent, warp-specialised, TMA-staged FFMA2
//   blend of the group records (described at the kernel).
// blend_kernel    -- D % 4 != 0 (D <= 128): CTA = one tile, warp = one pixel group at a time, feature rows loaded once per
//   record and applied to the 8 pixels of the group from registers; epilogue x 1/(1 - T^Q) (line 20), streaming stores.
#include "qr_async.cuh"
#include "qr_blend.cuh"

namespace qr {

constexpr int kWalkThreads = 256;
constexpr int kWalkBatch = 256;

// workspace layout: tile ticket, gcount[G], ucount[2 T], rec[G][cap] (G = tiles * 32 groups, cap = 8 K + kSentinels).
// Records are described in qr_blend.cuh.  Each list ends with kSentinels records of id -1 / weight 0 so that the
// FFMA blend pipeline can prefetch past the end.
struct FwdLayout {
    size_t ticket, gcount, ucount, rec, total;
    int64_t G;
    int cap;
    SelLayout sel;       // selection lists of the tcgen05 path (qr_sel.cuh); they share the region of the group records
};

static FwdLayout fwd_layout(const Cam& cam, int K)
{
    FwdLayout L;
    L.G = (int64_t)cam.tiles_x * cam.tiles_y * kGroupsPerTile;
    L.cap = kGroupPx * K + kSentinels;
    size_t o = 0;
    L.ticket = o; o = align_up(o + 4, 256);
    L.gcount = o; o = align_up(o + (size_t)L.G * 4, 256);
    L.ucount = o; o = align_up(o + (size_t)(L.G / 16) * 4, 256);
    L.rec = o;    o = align_up(o + (size_t)L.G * L.cap * kRecWords * 4, 256);
    const WsLayout wl = ws_layout(cam, K);      // tcgen05 path: the layout qr_backward_lists / qr_backward_clear also read
    L.sel = wl.sel;
    L.total = o > wl.total ? o : wl.total;
    return L;
}

struct WalkParams {
    Cam cam;
    int32_t K, cap;
    const float2* mean2d;
    const float4* conic_opac;
    const uint32_t* isect;
    const int2* tile_range;
    int32_t* n_sel;
    float* resid;
    int32_t* sel_idx;     // written here: used slots from the group records after the walk, then the -1 / 0 padding
    float* sel_w;
    int32_t* gcount;
    int32_t* ucount;      // [2 T] union size of each 16x8 half tile
    float* rec;
    int32_t* tile_ticket; // blend_kernel's tile queue, reset here
    int32_t batch_n = 0, view_h = 0;   // qr_forward_batch (see WalkParams2)
};

__global__ void __launch_bounds__(kWalkThreads, 5) walk_kernel(const WalkParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* ent_co = reinterpret_cast<float4*>(smem_raw);                 // [256] a, b, c, opacity
    float4* ent_box = ent_co + kWalkBatch;                                // [256] x_lo, x_hi, y_lo, y_hi
    float2* ent_xy = reinterpret_cast<float2*>(ent_box + kWalkBatch);     // [256]
    int32_t* ent_id = reinterpret_cast<int32_t*>(ent_xy + kWalkBatch);    // [256]
    float* thr = reinterpret_cast<float*>(ent_id + kWalkBatch);           // [K+1]
    __shared__ int32_t nsel_s[kTile * kTile];
    __shared__ int32_t ent_col[2][kWalkBatch];   // column of a batch entry in its half tile's union, -1 = not selected yet
    __shared__ int32_t ucount_s[2];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x;
    if (tile == 0 && tid == 0) *p.tile_ticket = 0;
    const int tile_x = tile % p.cam.tiles_x, tile_y = tile / p.cam.tiles_x;
    const int K = p.K;
    // warp = pixel rows 2*warp, 2*warp+1 of the tile; lane -> (x = lane & 15, y = lane >> 4)
    const int px = tile_x * kTile + (lane & 15), py = tile_y * kTile + warp * 2 + (lane >> 4);
    const bool inside = px < p.cam.width && py < p.cam.height;
    // batch of views stacked as one tall tile grid (qr_forward_batch): alpha' in the view's own pixel coordinates
    const int yoff = p.view_h > 0 ? (tile_y * kTile / p.view_h) * p.view_h : 0;
    const float fpx = (float)px + 0.5f, fpy = (float)(py - yoff) + 0.5f;          // R5
    const float wx_lo = (float)(tile_x * kTile), wx_hi = wx_lo + (float)kTile;
    const float wy_lo = (float)(tile_y * kTile - yoff + warp * 2), wy_hi = wy_lo + 2.0f;
    // group of this lane: gx = (lane & 15) >> 2 ; slot of the pixel inside its group q = (lane >> 4) * 4 + (lane & 3)
    const int gx = (lane & 15) >> 2, q = (lane >> 4) * 4 + (lane & 3);
    const uint32_t gbits = (0xFu << (4 * gx)) | (0xFu << (16 + 4 * gx));  // lanes of my group
    const int64_t group = (int64_t)tile * kGroupsPerTile + warp * 4 + gx;
    float* my_rec = p.rec + group * p.cap * kRecWords;

    for (int k = tid; k <= K; k += kWalkThreads)                          // thresholds as printed (R3)
        thr[k] = __fsub_rn(1.0f, __fdiv_rn((float)(k + 1), (float)(K + 1)));
    const float t_break = __fdiv_rn(1.0f, (float)(K + 1));
    const int2 range = p.tile_range[tile];
    const int half = warp >> 2;                                           // rows 0..7 / 8..15 of the tile
    if (tid < 2) ucount_s[tid] = 0;

    bool done = !inside;
    float T = 1.0f, TQ = 1.0f;
    int k = 0, ns = 0, gcnt = 0;
    bool warp_done = __all_sync(0xffffffffu, done);

    for (int b0 = range.x; b0 < range.y; b0 += kWalkBatch) {
        if (__syncthreads_and(warp_done)) break;                          // every pixel of the tile has stopped
        // ---- stage the batch ----
        {
            const int idx = b0 + tid;
            int32_t id = -1;
            float4 co = make_float4(0.f, 0.f, 0.f, 0.f), box = make_float4(1.f, 0.f, 1.f, 0.f);   // empty box
            float2 xy = make_float2(0.f, 0.f);
            if (idx < range.y) {
                id = (int32_t)p.isect[idx];
                xy = __ldg(p.mean2d + id);
                co = __ldg(p.conic_opac + id);
                // AABB of the 3-sigma ellipse recovered from the conic (cov = conic^-1), inflated so that fp32 rounding
                // can never drop a pixel that rule R4 includes
                const float det = co.x * co.z - co.y * co.y;
                float ex = 3.0e30f, ey = 3.0e30f;
                if (det > 0.0f) {
                    ex = 3.0f * sqrtf(co.z / det) * 1.001f + 0.01f;
                    ey = 3.0f * sqrtf(co.x / det) * 1.001f + 0.01f;
                }
                box = make_float4(xy.x - ex, xy.x + ex, xy.y - ey, xy.y + ey);
            }
            if (p.batch_n > 0 && id >= 0) id = (int32_t)((uint32_t)id % (uint32_t)p.batch_n);     // virtual Gaussian b N + i -> i
            ent_id[tid] = id; ent_co[tid] = co; ent_xy[tid] = xy; ent_box[tid] = box;
            ent_col[0][tid] = -1; ent_col[1][tid] = -1;
        }
        __syncthreads();
        if (warp_done) continue;
        const int nb = min(kWalkBatch, range.y - b0);

        // ---- entries whose box meets this warp's 16x2 pixels: 8 lane-parallel tests + ballots ----
        for (int c = 0; c < nb; c += 32) {
            const float4 box = ent_box[c + lane];
            uint32_t m = __ballot_sync(0xffffffffu, box.x < wx_hi && box.y > wx_lo && box.z < wy_hi && box.w > wy_lo);
            while (m) {
                const int e = c + __ffs(m) - 1;
                m &= m - 1;
                const float4 co = ent_co[e];
                const float2 xy = ent_xy[e];
                // alpha' (Eq. 1) with inclusion rule R4, fp32 decision arithmetic
                const float dx = __fsub_rn(fpx, xy.x), dy = __fsub_rn(fpy, xy.y);
                const float q1 = __fmul_rn(__fmul_rn(co.x, dx), dx);
                const float q2 = __fmaf_rn(__fmul_rn(co.z, dy), dy, q1);
                const float q3 = __fmul_rn(__fmul_rn(co.y, dx), dy);
                const float power = __fmaf_rn(-0.5f, q2, -q3);
                bool sel = false;
                float wQ = 0.0f;
                if (!done && !(power > 0.0f) && !(power < kPowerMin)) {
                    const float a = fminf(kAlphaMax, __fmul_rn(co.w, expf(power)));
                    if (!(a < kAlphaMin)) {
                        const float T_test = __fmul_rn(T, __fsub_rn(1.0f, a));          // line 5
                        if (T_test < thr[k]) {                                          // line 6
                            k = k + 1;                                                  // line 7
                            wQ = __fmul_rn(TQ, a);                                      // line 8
                            sel = true;                                                 // line 9 runs in blend_kernel
                            ++ns;
                            TQ = __fmul_rn(TQ, __fsub_rn(1.0f, a));                     // line 10
                            while (T_test < thr[k]) k = k + 1;                          // lines 11-13
                        }
                        if (T_test < t_break) done = true;                              // lines 15-17
                        else T = T_test;                                                // line 18
                    }
                }
                const uint32_t sm = __ballot_sync(0xffffffffu, sel);
                if (sm) {
                    // column of this Gaussian in the half tile's union: the first warp to select it numbers it
                    int col = 0;
                    if (lane == 0) {
                        volatile int32_t* slot = &ent_col[half][e];
                        const int old = atomicCAS(&ent_col[half][e], -1, -2);
                        if (old == -1) { col = atomicAdd(&ucount_s[half], 1); *slot = col; }
                        else { col = old; while (col == -2) col = *slot; }
                    }
                    col = __shfl_sync(0xffffffffu, col, 0);
                    if (sm & gbits) {                       // some pixel of my group selected this Gaussian
                        my_rec[gcnt * kRecWords + q] = wQ;  // 8 lanes write the record's 8 weights (32 contiguous bytes)
                        if (q == 0) {
                            // word 8 = Gaussian id, word 9 = which of the 8 pixels selected it (bit q) | column << 8
                            const uint32_t nz = ((sm >> (4 * gx)) & 0xFu) | (((sm >> (16 + 4 * gx)) & 0xFu) << 4);
                            *reinterpret_cast<float2*>(my_rec + gcnt * kRecWords + 8) =
                                make_float2(__int_as_float(ent_id[e]), __int_as_float((int)(nz | ((uint32_t)col << 8))));
                        }
                        ++gcnt;
                    }
                }
            }
            if (__all_sync(0xffffffffu, done)) { warp_done = true; break; }
        }
    }

    if (q == 0) p.gcount[group] = gcnt;
#pragma unroll
    for (int t = 0; t < kSentinels; ++t) {              // list terminators: weight 0, id -1
        my_rec[(gcnt + t) * kRecWords + q] = 0.0f;
        if (q == 0) my_rec[(gcnt + t) * kRecWords + 8] = __int_as_float(-1);
    }
    if (inside) {
        const int64_t pix = (int64_t)py * p.cam.width + px;
        p.n_sel[pix] = ns;
        p.resid[pix] = ns > 0 ? TQ : 1.0f;              // R8
    }
    // ---- selection records of the used slots, from the four group lists this warp has just written: lane = record,
    // a ballot per pixel ranks the records that selected it (its slot, depth order), weight x 1 / (1 - T^Q) (line 20).
    // Done here, at full occupancy, rather than by the W builders of the persistent blend kernel, whose ~1,100
    // dependent instructions per build were that kernel's critical path (profiles/README.md, r1_e). ----
    {
        const float inv = ns > 0 ? __fdiv_rn(1.0f, __fsub_rn(1.0f, TQ)) : 0.0f;
        const uint32_t lt_mask = (1u << lane) - 1u;
        __syncwarp();
#pragma unroll 1
        for (int g4 = 0; g4 < 4; ++g4) {
            const int n = __shfl_sync(0xffffffffu, gcnt, g4 * 4);                   // lane g4 * 4 belongs to group g4
            const float* recs = p.rec + ((int64_t)tile * kGroupsPerTile + warp * 4 + g4) * p.cap * kRecWords;
            int base[kGroupPx];
#pragma unroll
            for (int j = 0; j < kGroupPx; ++j) base[j] = 0;
            for (int i0 = 0; i0 < n; i0 += 32) {
                const int i = i0 + lane;
                const bool have = i < n;
                float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
                float2 m2 = make_float2(0.f, 0.f);
                if (have) {
                    a = *reinterpret_cast<const float4*>(recs + (size_t)i * kRecWords);
                    b = *reinterpret_cast<const float4*>(recs + (size_t)i * kRecWords + 4);
                    m2 = *reinterpret_cast<const float2*>(recs + (size_t)i * kRecWords + 8);
                }
                const float w[kGroupPx] = { a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w };
                const int32_t id = __float_as_int(m2.x);
                const uint32_t nz = have ? ((uint32_t)__float_as_int(m2.y) & 0xFFu) : 0u;
#pragma unroll
                for (int j = 0; j < kGroupPx; ++j) {
                    const bool bit = (nz >> j) & 1u;
                    const uint32_t bal = __ballot_sync(0xffffffffu, bit);
                    const int pl = (j >> 2) * 16 + g4 * 4 + (j & 3);                 // lane that owns pixel j of group g4
                    const float inv_j = __shfl_sync(0xffffffffu, inv, pl);
                    const int qx = tile_x * kTile + (pl & 15), qy = tile_y * kTile + warp * 2 + (pl >> 4);
                    if (bit && qx < p.cam.width && qy < p.cam.height) {
                        const int64_t o = ((int64_t)qy * p.cam.width + qx) * K + base[j] + __popc(bal & lt_mask);
                        p.sel_idx[o] = id;
                        p.sel_w[o] = __fmul_rn(w[j], inv_j);
                    }
                    base[j] += __popc(bal);
                }
            }
        }
    }
    // ---- padding of the selection records (-1 / 0 for slots >= n_sel), coalesced: a tile row is 16*K contiguous
    // words of sel_idx / sel_w. ----
    nsel_s[warp * 32 + lane] = ns;                      // index = (2*warp + (lane>>4))*16 + (lane&15) = y_local*16 + x_local
    __syncthreads();
    if (tid < 2) p.ucount[tile * 2 + tid] = ucount_s[tid];
    {
        const int npx = min(kTile, p.cam.width - tile_x * kTile);
        const int row_words = npx * K;
        const int dq = kWalkThreads / K, dr = kWalkThreads % K;      // advancing i by 256 = dq pixels and dr slots
        for (int r = 0; r < kTile; ++r) {
            const int y = tile_y * kTile + r;
            if (y >= p.cam.height) break;
            const int64_t gbase = ((int64_t)y * p.cam.width + tile_x * kTile) * K;
            int pxl = tid / K, sl = tid - pxl * K;
            for (int i = tid; i < row_words; i += kWalkThreads) {
                if (sl >= nsel_s[r * kTile + pxl]) {
                    p.sel_idx[gbase + i] = -1;
                    p.sel_w[gbase + i] = 0.0f;
                }
                pxl += dq; sl += dr;
                if (sl >= K) { sl -= K; ++pxl; }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------

template <typename FeatT, int VW> struct Row;
template <> struct Row<float, 4> {
    static __device__ __forceinline__ void load(const float* src, float (&f)[4])
    {
        const float4 v = __ldg(reinterpret_cast<const float4*>(src));
        f[0] = v.x; f[1] = v.y; f[2] = v.z; f[3] = v.w;
    }
};
template <> struct Row<float, 1> {
    static __device__ __forceinline__ void load(const float* src, float (&f)[1]) { f[0] = __ldg(src); }
};
template <> struct Row<__half, 8> {
    static __device__ __forceinline__ void load(const __half* src, float (&f)[8])
    {
        const uint4 v = __ldg(reinterpret_cast<const uint4*>(src));
        const __half2* h = reinterpret_cast<const __half2*>(&v);
#pragma unroll
        for (int i = 0; i < 4; ++i) { const float2 t = __half22float2(h[i]); f[2 * i] = t.x; f[2 * i + 1] = t.y; }
    }
};

template <int VW> __device__ __forceinline__ void store_map(float* dst, const float (&v)[VW]);
template <> __device__ __forceinline__ void store_map<4>(float* dst, const float (&v)[4])
{
    __stcs(reinterpret_cast<float4*>(dst), make_float4(v[0], v[1], v[2], v[3]));
}
template <> __device__ __forceinline__ void store_map<1>(float* dst, const float (&v)[1]) { __stcs(dst, v[0]); }
template <> __device__ __forceinline__ void store_map<8>(float* dst, const float (&v)[8])
{
    __stcs(reinterpret_cast<float4*>(dst), make_float4(v[0], v[1], v[2], v[3]));
    __stcs(reinterpret_cast<float4*>(dst) + 1, make_float4(v[4], v[5], v[6], v[7]));
}

constexpr int kBlendWarps = 8;
constexpr int kBlendSlots = 64;              // ring of tiles a CTA has claimed (only ~2 are live at any time)


// Persistent CTAs (one per SM).  Work is handed out without block barriers: a warp takes a ticket from the CTA's
// shared counter; ticket / 32 is a slot of the CTA's tile ring, ticket % 32 the pixel group inside that tile.  The
// warp that draws group 0 of a slot claims the next tile from the global queue and publishes it; the others wait
// for that word only.  All warps of a CTA therefore work on the same one or two tiles (feature rows shared by the
// tile's groups stay in L1) and nobody idles at a barrier when group list lengths differ.
template <typename FeatT, int NV, int VW, bool FULL>
__global__ void __launch_bounds__(kBlendWarps * 32, 1) blend_kernel(const BlendParams p)
{
    __shared__ int32_t s_ticket;
    __shared__ unsigned long long s_slot[kBlendSlots];   // ((slot + 1) << 32) | tile, 0 = never written
    __shared__ int32_t s_reads[kBlendSlots];             // how many of the slot's 31 other groups have read it
    const int lane = threadIdx.x & 31;
    const int D = p.D;
    if (threadIdx.x == 0) s_ticket = 0;
    if (threadIdx.x < kBlendSlots) { s_slot[threadIdx.x] = 0ull; s_reads[threadIdx.x] = 0; }
    __syncthreads();

    // ---- work hand-out ----
    struct Job { int tile, g, n; int32_t ids0, ids1; float inv; };   // inv: lanes 0..7 = 1/(1 - T^Q) of pixel q = lane
    auto draw = [&](Job& jb) {
        // next (tile, group) of this CTA; groups outside the image are skipped; tile >= num_tiles means "no more work".
        // The loads every record of the group's list depends on (count, first 64 ids, T^Q) are issued here, one group
        // ahead of their use.
        while (true) {
            int tile = 0, g = 0;
            if (lane == 0) {
                const int ticket = atomicAdd(&s_ticket, 1);
                const int slot = ticket >> 5, idx = slot % kBlendSlots;
                g = ticket & 31;
                volatile unsigned long long* word = &s_slot[idx];
                volatile int32_t* reads = &s_reads[idx];
                if (g == 0) {
                    // claim the next tile for this slot.  The ring entry is reused every kBlendSlots tiles: wait until
                    // the 31 readers of its previous generation are through (they never wait on this warp: this ends)
                    if (slot >= kBlendSlots) { while (*reads != 31) { } }
                    *reads = 0;
                    tile = atomicAdd(p.tile_ticket, 1);
                    __threadfence_block();
                    *word = ((unsigned long long)(slot + 1) << 32) | (unsigned int)tile;
                } else {
                    unsigned long long v;
                    while (((v = *word) >> 32) != (unsigned long long)(slot + 1)) { }
                    tile = (int)(v & 0xffffffffull);
                    atomicAdd(&s_reads[idx], 1);
                }
            }
            jb.tile = __shfl_sync(0xffffffffu, tile, 0);
            jb.g = __shfl_sync(0xffffffffu, g, 0);
            if (jb.tile >= p.num_tiles) return;
            const int gx0 = (jb.tile % p.cam.tiles_x) * kTile + (jb.g & 3) * 4;
            const int gy0 = (jb.tile / p.cam.tiles_x) * kTile + (jb.g >> 2) * 2;
            if (gx0 >= p.cam.width || gy0 >= p.cam.height) continue;
            const int64_t group = (int64_t)jb.tile * kGroupsPerTile + jb.g;
            const float* rec = p.rec + group * p.cap * kRecWords;
            jb.n = __ldg(p.gcount + group);
            // ids of records lane and 32 + lane (inside the group's capacity whenever K >= 8; guarded otherwise)
            jb.ids0 = lane < p.cap ? __float_as_int(__ldg(rec + lane * kRecWords + 8)) : -1;
            jb.ids1 = lane + 32 < p.cap ? __float_as_int(__ldg(rec + (lane + 32) * kRecWords + 8)) : -1;
            const int mx = gx0 + (lane & 3), my = gy0 + ((lane >> 2) & 1);
            jb.inv = 0.0f;
            if (lane < kGroupPx && mx < p.cam.width && my < p.cam.height) {
                const int64_t mpix = (int64_t)my * p.cam.width + mx;
                if (__ldg(p.n_sel + mpix) > 0) jb.inv = __fdiv_rn(1.0f, __fsub_rn(1.0f, __ldg(p.resid + mpix)));   // line 20; R8
            }
            return;
        }
    };

    Job cur, nxt;
    draw(cur);
    while (cur.tile < p.num_tiles) {
        draw(nxt);
        const int tile = cur.tile, g = cur.g, n = cur.n;
        const int tile_x = tile % p.cam.tiles_x, tile_y = tile / p.cam.tiles_x;
        // group g = (row pair g >> 2, x block g & 3); pixel q of the group: x = 4*(g&3) + (q&3), y = 2*(g>>2) + (q>>2)
        const int gx0 = tile_x * kTile + (g & 3) * 4, gy0 = tile_y * kTile + (g >> 2) * 2;
        const int64_t group = (int64_t)tile * kGroupsPerTile + g;
        const float* recf = p.rec + group * p.cap * kRecWords;
        const float4* rec4 = reinterpret_cast<const float4*>(recf);
        const float* recw = recf + (lane & 7);                               // lane q < 8: its own pixel's weight

        // lanes 0..7 carry 1/(1 - T^Q) of pixel q = lane
        const float minv = cur.inv;

        float acc[kGroupPx][NV][VW];
#pragma unroll
        for (int q = 0; q < kGroupPx; ++q)
#pragma unroll
            for (int j = 0; j < NV; ++j)
#pragma unroll
                for (int v = 0; v < VW; ++v) acc[q][j][v] = 0.0f;

        // Software pipeline over three register sets: while record i is applied, the feature rows of records i+1 and
        // i+2 and the weights of record i+3 are in flight.  Ids come from the lane-parallel prefetch (ids0 = records
        // 32b..32b+31 of the current block b, ids1 = the next block), so a row load never waits for its id.
        int32_t ids0 = cur.ids0, ids1 = cur.ids1;
        int blk = 0;
        auto id_at = [&](int i) -> int32_t {           // i in block blk or blk + 1; -1 past the end of the list
            const int32_t v = __shfl_sync(0xffffffffu, ((i >> 5) == blk) ? ids0 : ids1, i & 31);
            return i < n ? v : -1;
        };
        struct Meta { float4 w0, w1; float wm; };
        auto load_meta = [&](int i) {
            Meta m;
            m.w0 = __ldg(rec4 + 3 * i);
            m.w1 = __ldg(rec4 + 3 * i + 1);
            m.wm = __ldg(recw + (size_t)i * kRecWords);
            return m;
        };
        auto load_row = [&](int32_t id, float (&f)[NV][VW]) {
            if (id >= 0) {
                const FeatT* rowp = static_cast<const FeatT*>(p.features) + (int64_t)id * D + lane * VW;
#pragma unroll
                for (int j = 0; j < NV; ++j) {
                    if (FULL || (j * 32 + lane) * VW < D) Row<FeatT, VW>::load(rowp + j * 32 * VW, f[j]);
                    else {
#pragma unroll
                        for (int v = 0; v < VW; ++v) f[j][v] = 0.0f;
                    }
                }
            }
        };
        auto apply = [&](const Meta& m, int32_t id, const float (&f)[NV][VW]) {
            // which of the 8 pixels selected this Gaussian: a ballot, so the branches below are provably uniform
            const uint32_t nz = __ballot_sync(0xffffffffu, m.wm != 0.0f) & 0xFFu;
            const float w[kGroupPx] = { m.w0.x, m.w0.y, m.w0.z, m.w0.w, m.w1.x, m.w1.y, m.w1.z, m.w1.w };
#pragma unroll
            for (int q = 0; q < kGroupPx; ++q) {
                if (nz & (1u << q)) {
#pragma unroll
                    for (int j = 0; j < NV; ++j)
#pragma unroll
                        for (int v = 0; v < VW; ++v) acc[q][j][v] = __fmaf_rn(w[q], f[j][v], acc[q][j][v]);   // line 9
                }
            }
        };
        float fA[NV][VW], fB[NV][VW], fC[NV][VW];
        int32_t iA = id_at(0), iB = id_at(1), iC = id_at(2);
        Meta mA = load_meta(0), mB = load_meta(1), mC = load_meta(2);
        load_row(iA, fA);
        load_row(iB, fB);
        for (int i = 0; i < n; i += 3) {
            if (((i + 5) >> 5) > blk + 1) {            // the pipeline is about to leave block blk + 1: slide the id window
                ++blk;
                ids0 = ids1;
                const int r = (blk + 1) * 32 + lane;
                ids1 = r < p.cap ? __float_as_int(__ldg(recf + (size_t)r * kRecWords + 8)) : -1;
            }
            load_row(iC, fC);
            { const Meta m = mA; const int32_t id = iA; mA = load_meta(i + 3); iA = id_at(i + 3); apply(m, id, fA); }
            if (i + 1 >= n) break;
            load_row(iA, fA);
            { const Meta m = mB; const int32_t id = iB; mB = load_meta(i + 4); iB = id_at(i + 4); apply(m, id, fB); }
            if (i + 2 >= n) break;
            load_row(iB, fB);
            { const Meta m = mC; const int32_t id = iC; mC = load_meta(i + 5); iC = id_at(i + 5); apply(m, id, fC); }
        }

        // ---- epilogue: normalise and store (512 contiguous bytes per store instruction) ----
#pragma unroll
        for (int q = 0; q < kGroupPx; ++q) {
            const int x = gx0 + (q & 3), y = gy0 + (q >> 2);
            const float inv = __shfl_sync(0xffffffffu, minv, q);
            if (x < p.cam.width && y < p.cam.height) {
                float* dst = p.out_map + ((int64_t)y * p.cam.width + x) * D;
#pragma unroll
                for (int j = 0; j < NV; ++j) {
                    const int ch = (j * 32 + lane) * VW;
                    if (FULL || ch < D) {
                        float o[VW];
#pragma unroll
                        for (int v = 0; v < VW; ++v) o[v] = __fmul_rn(acc[q][j][v], inv);
                        store_map<VW>(dst + ch, o);
                    }
                }
            }
        }
        cur = nxt;
    }
}

// ---------------------------------------------------------------------------------------------------------------
// blend_tu_kernel -- the O(KC) blend with the band's union of selected Gaussians staged ONCE in shared memory by TMA.
//
// Persistent CTA = 1 producer warp + 8 consumer warps.  Work item = one 16x4-pixel band of a tile = 8 pixel groups,
// one per consumer warp.  The producer builds a stage: it takes up to kTuRecs records of each of the band's 8 lists,
// numbers the distinct Gaussian ids among them (shared-memory hash set), and issues one bulk async copy
// (cp.async.bulk ... mbarrier::complete_tx) per distinct feature row and per record list into the stage buffers.
// Consumers wait on the stage's "full" mbarrier, then read weights, row slots and rows from shared memory only:
// a feature row crosses L2 -> SM once per band instead of once per pixel group, and no consumer ever waits on a
// global load.  Two stages: the producer fills one while the consumers drain the other.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kTuConsumers = 8;
constexpr int kTuProducers = 4;        // warps 8..11, one per scheduler
constexpr int kTuThreads = 384;         // warps 0..7 consumers, warps 8..11 producers
constexpr int kTuProducerRegs = 72;    // setmaxnreg: 12 warps start at 168 registers; the producer warpgroup drops to
constexpr int kTuConsumerRegs = 216;   // 72 and the two consumer warpgroups grow to 216 (128 accumulators + 2 row sets)
constexpr int kTuStages = 2;
constexpr int kTuRows = 46;            // distinct feature rows per stage
constexpr int kTuRecs = 32;            // records per group per stage (one per producer lane)
constexpr int kTuHash = 512;           // >= 2 * 8 * kTuRecs

struct TuDesc {
    int32_t tile, band, flags;         // flags: 1 = first stage of the band, 2 = last stage, 4 = no more work
    int32_t nrec[kTuConsumers];
    float inv[kTuConsumers * kGroupPx];   // 1/(1 - T^Q) per pixel of the band, 0 where nothing is selected
};

using namespace aq;     // mbarrier / bulk-copy helpers (qr_async.cuh)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return s32(p); }

template <typename FeatT, int VW> struct SRow;
template <> struct SRow<float, 4> {
    static __device__ __forceinline__ void load(const unsigned char* row, int lane_vec, float (&f)[4])
    {
        const float4 v = *reinterpret_cast<const float4*>(row + (size_t)lane_vec * 16);
        f[0] = v.x; f[1] = v.y; f[2] = v.z; f[3] = v.w;
    }
};
template <> struct SRow<__half, 8> {
    static __device__ __forceinline__ void load(const unsigned char* row, int lane_vec, float (&f)[8])
    {
        const uint4 v = *reinterpret_cast<const uint4*>(row + (size_t)lane_vec * 16);
        const __half2* h = reinterpret_cast<const __half2*>(&v);
#pragma unroll
        for (int i = 0; i < 4; ++i) { const float2 t = __half22float2(h[i]); f[2 * i] = t.x; f[2 * i + 1] = t.y; }
    }
};

struct TuSmem {            // offsets into dynamic shared memory
    int rows, recs, rslot, desc, bars, hkey, hslot, uniq, total;
};
__host__ __device__ inline TuSmem tu_smem(int rowbytes)
{
    TuSmem L;
    int o = 0;
    L.rows = o;  o += kTuStages * kTuRows * rowbytes;
    L.recs = o;  o += kTuStages * kTuConsumers * kTuRecs * kRecWords * 4;
    L.desc = o;  o += (kTuStages * (int)sizeof(TuDesc) + 15) & ~15;
    L.bars = o;  o += 2 * kTuStages * 8;
    L.hkey = o;  o += kTuProducers * kTuHash * 4;
    L.uniq = o;  o += kTuProducers * 48 * 4;
    L.rslot = o; o += kTuStages * kTuConsumers * kTuRecs;
    L.hslot = o; o += kTuProducers * kTuHash;
    L.total = (o + 15) & ~15;
    return L;
}

template <typename FeatT, int NV, int VW, bool FULL>
__global__ void __launch_bounds__(kTuThreads, 1) blend_tu_kernel(const BlendParams p)
{
    extern __shared__ __align__(128) unsigned char smem[];
    const int D = p.D;
    const int rowbytes = D * (int)sizeof(FeatT);
    const TuSmem L = tu_smem(rowbytes);
    unsigned char* s_rows = smem + L.rows;
    float* s_recs = reinterpret_cast<float*>(smem + L.recs);
    TuDesc* s_desc = reinterpret_cast<TuDesc*>(smem + L.desc);
    uint64_t* s_full = reinterpret_cast<uint64_t*>(smem + L.bars);
    uint64_t* s_empty = s_full + kTuStages;
    uint8_t* s_rslot = smem + L.rslot;
    __shared__ int32_t s_lock, s_it, s_finished;   // producers: publish lock, next stage number, producers out of work

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        s_lock = 0; s_it = 0; s_finished = 0;
        for (int s = 0; s < kTuStages; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], kTuConsumers); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int num_items = p.num_tiles * 4;

    if (warp >= kTuConsumers) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kTuProducerRegs));
        // =========================================== producers ===========================================
        // Four producer warps, one per scheduler, each building the stages of its own bands: a producer warp shares
        // its scheduler with two consumer warps that issue FFMAs back to back, so one stage build takes ~20k cycles
        // of wall time (measured) although it is a few hundred instructions; four bands in flight keep the stage
        // rate above what the consumers drain.  Publishing (wait for a free buffer, descriptor, copies) is
        // serialised by a lock so that the stages of one band stay contiguous and in order.
        const int pw = warp - kTuConsumers;
        int32_t* s_hkey = reinterpret_cast<int32_t*>(smem + L.hkey) + pw * kTuHash;
        int32_t* s_uniq = reinterpret_cast<int32_t*>(smem + L.uniq) + pw * 48;
        uint8_t* s_hslot = smem + L.hslot + pw * kTuHash;
        volatile int32_t* v_it = &s_it;
        // Per item (band) the producer needs the 8 list lengths and the 64 pixels' T^Q; those loads, and the ticket
        // itself, are issued one item ahead so that their latency hides behind the stage building of the current item.
        struct Item { int item; int n_w; float inv2[2]; };
        auto fetch = [&](Item& t) {
            int item = 0;
            if (lane == 0) item = atomicAdd(p.tile_ticket, 1);
            t.item = __shfl_sync(0xffffffffu, item, 0);
            t.n_w = 0; t.inv2[0] = t.inv2[1] = 0.0f;
            if (t.item >= num_items) return;
            const int tile = t.item >> 2, band = t.item & 3;
            const int x0 = (tile % p.cam.tiles_x) * kTile, y0 = (tile / p.cam.tiles_x) * kTile + band * 4;
            if (y0 >= p.cam.height) return;
            t.n_w = __ldg(p.gcount + (int64_t)tile * kGroupsPerTile + band * 8 + (lane & 7));
#pragma unroll
            for (int h = 0; h < 2; ++h) {      // lane handles pixels lane and lane + 32 of the band (group-major numbering)
                const int gp = lane + 32 * h, w = gp >> 3, q = gp & 7;
                const int x = x0 + (w & 3) * 4 + (q & 3), y = y0 + (w >> 2) * 2 + (q >> 2);
                if (x < p.cam.width && y < p.cam.height) {
                    const int64_t pix = (int64_t)y * p.cam.width + x;
                    if (__ldg(p.n_sel + pix) > 0) t.inv2[h] = __fdiv_rn(1.0f, __fsub_rn(1.0f, __ldg(p.resid + pix)));   // line 20; R8
                }
            }
        };
        auto lock = [&]() {
            if (lane == 0) { while (atomicCAS(&s_lock, 0, 1) != 0) { } }
            __syncwarp();
            __threadfence_block();
        };
        auto unlock = [&]() {
            __threadfence_block();
            __syncwarp();
            if (lane == 0) atomicExch(&s_lock, 0);
        };
        Item cur_item, next_item;
        fetch(cur_item);
        while (true) {
            const int item = cur_item.item;
            if (item >= num_items) {
                // the last producer to run out of work tells the consumers to stop
                int last_one = 0;
                if (lane == 0) last_one = atomicAdd(&s_finished, 1) == kTuProducers - 1;
                if (__shfl_sync(0xffffffffu, last_one, 0)) {
                    lock();
                    const int it = *v_it;
                    const int s_done = it % kTuStages;
                    mbar_wait(&s_empty[s_done], ((it / kTuStages) & 1) ^ 1);
                    if (lane == 0) { s_desc[s_done].flags = 4; mbar_arrive(&s_full[s_done]); }
                    unlock();
                }
                break;
            }
            fetch(next_item);
            const int tile = item >> 2, band = item & 3;
            const int y0 = (tile / p.cam.tiles_x) * kTile + band * 4;
            if (y0 >= p.cam.height) { cur_item = next_item; continue; }   // band below the image: nothing to render
            // lane w < 8 tracks group w of the band: list length and progress
            const int64_t gi = (int64_t)tile * kGroupsPerTile + band * 8 + (lane & 7);
            const int n_w = cur_item.n_w;
            int r0_w = 0;
            const float inv2[2] = { cur_item.inv2[0], cur_item.inv2[1] };
            bool first = true, locked = false;
            while (true) {
                // ---- choose the stage's records: up to R per group such that their distinct rows fit ----
                int R = kTuRecs, cnt_w = 0, U = 0;
                int32_t ids[kTuConsumers];
                uint8_t slot8[kTuConsumers];
                int hcell[kTuConsumers];
                while (true) {
                    cnt_w = min(R, n_w - r0_w);
                    for (int i = lane; i < kTuHash; i += 32) s_hkey[i] = -1;
                    __syncwarp();
#pragma unroll
                    for (int w = 0; w < kTuConsumers; ++w) {       // group w, record r0 + lane: 8 independent loads
                        const int c = __shfl_sync(0xffffffffu, cnt_w, w), r0 = __shfl_sync(0xffffffffu, r0_w, w);
                        ids[w] = -1;
                        if (lane < c) {
                            const int64_t g = (int64_t)tile * kGroupsPerTile + band * 8 + w;
                            ids[w] = __float_as_int(__ldg(p.rec + (g * p.cap + r0 + lane) * kRecWords + 8));
                        }
                    }
                    // insert: first probes of the 8 records are independent shared-memory CAS operations (in flight
                    // together); only collisions walk on
                    int32_t old[kTuConsumers];
#pragma unroll
                    for (int w = 0; w < kTuConsumers; ++w) {
                        hcell[w] = (int)(((uint32_t)ids[w] * 2654435761u) >> 23);       // 9 bits
                        old[w] = ids[w];
                        if (ids[w] >= 0) old[w] = atomicCAS(&s_hkey[hcell[w]], -1, ids[w]);
                    }
#pragma unroll
                    for (int w = 0; w < kTuConsumers; ++w) {
                        if (ids[w] >= 0 && old[w] != -1 && old[w] != ids[w]) {
                            int h = hcell[w];
                            while (true) {
                                h = (h + 1) & (kTuHash - 1);
                                const int32_t o = atomicCAS(&s_hkey[h], -1, ids[w]);
                                if (o == -1 || o == ids[w]) break;
                            }
                            hcell[w] = h;
                        }
                    }
                    __syncwarp();
                    // number the occupied cells with ballots (no atomics): cell i of lane-strided chunk c gets
                    // base + (occupied cells before it in the chunk)
                    U = 0;
#pragma unroll 4
                    for (int c = 0; c < kTuHash; c += 32) {
                        const int32_t id = s_hkey[c + lane];
                        const uint32_t occ = __ballot_sync(0xffffffffu, id >= 0);
                        if (id >= 0) {
                            const int slot = U + __popc(occ & ((1u << lane) - 1u));
                            s_hslot[c + lane] = (uint8_t)slot;
                            if (slot < kTuRows) s_uniq[slot] = id;
                        }
                        U += __popc(occ);
                    }
                    __syncwarp();
                    if (U <= kTuRows) break;
                    R = max(R >> 1, 1);                            // R = 1 always fits (<= 8 rows)
                }
#pragma unroll
                for (int w = 0; w < kTuConsumers; ++w) slot8[w] = ids[w] >= 0 ? s_hslot[hcell[w]] : (uint8_t)0;
                const bool last = __all_sync(0xffffffffu, r0_w + cnt_w >= n_w);

                // ---- publish the stage ----
                if (!locked) { lock(); locked = true; }
                const int it = *v_it;
                const int s = it % kTuStages;
                mbar_wait(&s_empty[s], ((it / kTuStages) & 1) ^ 1);
                TuDesc* d = &s_desc[s];
                if (lane == 0) { d->tile = tile; d->band = band; d->flags = (first ? 1 : 0) | (last ? 2 : 0); }
                if (lane < kTuConsumers) d->nrec[lane] = cnt_w;
                d->inv[lane] = inv2[0];
                d->inv[lane + 32] = inv2[1];
#pragma unroll
                for (int w = 0; w < kTuConsumers; ++w) s_rslot[(s * kTuConsumers + w) * kTuRecs + lane] = slot8[w];
                uint32_t bytes = (lane < kTuConsumers ? (uint32_t)cnt_w * kRecWords * 4u : 0u);
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) bytes += __shfl_xor_sync(0xffffffffu, bytes, o);
                bytes += (uint32_t)U * (uint32_t)rowbytes;
                __syncwarp();
                if (lane == 0) mbar_arrive_expect_tx(&s_full[s], bytes);
                __syncwarp();
                for (int u = lane; u < U; u += 32)
                    bulk_g2s(s_rows + ((size_t)s * kTuRows + u) * rowbytes,
                             static_cast<const unsigned char*>(p.features) + (size_t)s_uniq[u] * rowbytes,
                             (uint32_t)rowbytes, &s_full[s]);
                if (lane < kTuConsumers && cnt_w > 0)
                    bulk_g2s(s_recs + ((size_t)s * kTuConsumers + lane) * kTuRecs * kRecWords,
                             p.rec + (gi * p.cap + r0_w) * kRecWords, (uint32_t)cnt_w * kRecWords * 4u, &s_full[s]);
                __syncwarp();                        // s_uniq / s_hkey are rewritten by the next stage
                r0_w += cnt_w;
                first = false;
                if (lane == 0) *v_it = it + 1;
                if (last) break;
            }
            unlock();
            cur_item = next_item;
        }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kTuConsumerRegs));
        // =========================================== consumers ===========================================
        float2 acc[kGroupPx][NV][VW / 2];     // packed pairs: the blend runs on FFMA2 (fma.rn.f32x2)
        float minv = 0.0f;
        int gx0 = 0, gy0 = 0;
        for (int it = 0;; ++it) {
            const int s = it % kTuStages;
            mbar_wait(&s_full[s], (it / kTuStages) & 1);
            const TuDesc* d = &s_desc[s];
            const int flags = d->flags;
            if (flags & 4) break;
            if (flags & 1) {
                const int tile = d->tile, band = d->band;
                gx0 = (tile % p.cam.tiles_x) * kTile + (warp & 3) * 4;
                gy0 = (tile / p.cam.tiles_x) * kTile + band * 4 + (warp >> 2) * 2;
                minv = d->inv[warp * kGroupPx + (lane & 7)];
#pragma unroll
                for (int q = 0; q < kGroupPx; ++q)
#pragma unroll
                    for (int j = 0; j < NV; ++j)
#pragma unroll
                        for (int v = 0; v < VW / 2; ++v) acc[q][j][v] = make_float2(0.0f, 0.0f);
            }
            const int n = d->nrec[warp];
            const float* recs = s_recs + ((size_t)s * kTuConsumers + warp) * kTuRecs * kRecWords;
            const uint8_t* rslot = s_rslot + (s * kTuConsumers + warp) * kTuRecs;
            const unsigned char* rows = s_rows + (size_t)s * kTuRows * rowbytes;
            // Branch-free inner loop.  Measured on B200 (profiles/): with two warps per scheduler a predicated branch
            // costs a warp ~15-20 issue cycles, more than the 16 FFMAs it would skip, so all 8 pixels are always
            // updated (a pixel that did not select the Gaussian has weight 0).  Software pipeline over two register
            // sets: the weights / id / row of record i+1 are loaded from shared memory while record i is applied.
            struct Meta { float4 w0, w1; float wm; int32_t id; };
            auto load_meta = [&](int i) {
                Meta m;
                m.w0 = *reinterpret_cast<const float4*>(recs + i * kRecWords);
                m.w1 = *reinterpret_cast<const float4*>(recs + i * kRecWords + 4);
                m.id = __float_as_int(recs[i * kRecWords + 8]);
                m.wm = recs[i * kRecWords + (lane & 7)];
                return m;
            };
            auto load_f = [&](int i, float (&f)[NV][VW]) {
                const unsigned char* row = rows + (size_t)rslot[i] * rowbytes;
#pragma unroll
                for (int j = 0; j < NV; ++j) {
                    if (FULL || (j * 32 + lane) * VW < D) SRow<FeatT, VW>::load(row, j * 32 + lane, f[j]);
                    else {
#pragma unroll
                        for (int v = 0; v < VW; ++v) f[j][v] = 0.0f;
                    }
                }
            };
            auto apply = [&](const Meta& m, const float (&f)[NV][VW]) {
                const float w[kGroupPx] = { m.w0.x, m.w0.y, m.w0.z, m.w0.w, m.w1.x, m.w1.y, m.w1.z, m.w1.w };
#pragma unroll
                for (int q = 0; q < kGroupPx; ++q) {
                    const float2 ww = make_float2(w[q], w[q]);
#pragma unroll
                    for (int j = 0; j < NV; ++j)
#pragma unroll
                        for (int v = 0; v < VW / 2; ++v)       // line 9, two channels per instruction, each an IEEE fma
                            acc[q][j][v] = __ffma2_rn(ww, make_float2(f[j][2 * v], f[j][2 * v + 1]), acc[q][j][v]);
                }
            };
            if (n > 0) {
                float fA[NV][VW], fB[NV][VW];
                Meta mA = load_meta(0), mB;
                load_f(0, fA);
                int i = 0;
                for (; i + 1 < n; i += 2) {
                    mB = load_meta(i + 1); load_f(i + 1, fB);
                    apply(mA, fA);
                    if (i + 2 < n) { mA = load_meta(i + 2); load_f(i + 2, fA); }
                    apply(mB, fB);
                }
                if (n & 1) apply(mA, fA);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&s_empty[s]);     // stage buffers are free; the epilogue uses registers only
            if (flags & 2) {
#pragma unroll
                for (int q = 0; q < kGroupPx; ++q) {
                    const int x = gx0 + (q & 3), y = gy0 + (q >> 2);
                    const float inv = __shfl_sync(0xffffffffu, minv, q);
                    if (x < p.cam.width && y < p.cam.height) {
                        float* dst = p.out_map + ((int64_t)y * p.cam.width + x) * D;
#pragma unroll
                        for (int j = 0; j < NV; ++j) {
                            const int ch = (j * 32 + lane) * VW;
                            if (FULL || ch < D) {
                                float o[VW];
#pragma unroll
                                for (int v = 0; v < VW / 2; ++v) {
                                    o[2 * v] = __fmul_rn(acc[q][j][v].x, inv);
                                    o[2 * v + 1] = __fmul_rn(acc[q][j][v].y, inv);
                                }
                                store_map<VW>(dst + ch, o);
                            }
                        }
                    }
                }
            }
        }
    }
}

template <typename FeatT, int NV, int VW>
static int launch_blend_tu(const BlendParams& p, cudaStream_t st)
{
    const unsigned grid = (unsigned)min(sm_count(), p.num_tiles * 4);
    const int smem = tu_smem(p.D * (int)sizeof(FeatT)).total;
    if (p.D == NV * 32 * VW) {
        auto kern = blend_tu_kernel<FeatT, NV, VW, true>;
        QR_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        kern<<<grid, kTuThreads, smem, st>>>(p);
    } else {
        auto kern = blend_tu_kernel<FeatT, NV, VW, false>;
        QR_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        kern<<<grid, kTuThreads, smem, st>>>(p);
    }
    QR_LAUNCH_OK("blend_tu_kernel");
    return QR_OK;
}

template <typename FeatT, int NV, int VW>
static int launch_blend(const BlendParams& p, cudaStream_t st)
{
    const unsigned grid = (unsigned)min(sm_count(), p.num_tiles);
    if (p.D == NV * 32 * VW) blend_kernel<FeatT, NV, VW, true><<<grid, kBlendWarps * 32, 0, st>>>(p);
    else blend_kernel<FeatT, NV, VW, false><<<grid, kBlendWarps * 32, 0, st>>>(p);
    QR_LAUNCH_OK("blend_kernel");
    return QR_OK;
}

// blend_pixel_kernel -- D <= 8 with D % 4 != 0 (the RGB payload, D = 3): thread = pixel.  With so few channels a lane per
// channel (blend_kernel) leaves 29 of 32 lanes idle; here a thread walks its own selection record,
//     out[p,:] = sum_s sel_w[p,s] F[sel_idx[p,s],:]        (sel_w is already normalised by 1 - T^Q: line 20),
// the feature table (12 bytes per Gaussian) stays in L2, and a warp's 32 results leave as one contiguous 32 D-float block.
constexpr int kPixThreads = 256;
__global__ void __launch_bounds__(kPixThreads) blend_pixel_kernel(const BlendParams p)
{
    const int64_t pix = (int64_t)blockIdx.x * kPixThreads + threadIdx.x;
    if (pix >= (int64_t)p.cam.width * p.cam.height) return;
    const int D = p.D, K = p.K;
    const float* F = static_cast<const float*>(p.features);
    const int n = min(max(__ldg(p.n_sel + pix), 0), K);
    float acc[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) acc[c] = 0.0f;
    const int32_t* ids = p.sel_idx + pix * K;
    const float* ws = p.sel_w + pix * K;
    for (int s = 0; s < n; ++s) {
        const float w = ws[s];
        const float* f = F + (int64_t)ids[s] * D;
#pragma unroll
        for (int c = 0; c < 8; ++c)
            if (c < D) acc[c] = __fadd_rn(acc[c], __fmul_rn(w, __ldg(f + c)));
    }
    float* o = p.out_map + pix * D;
#pragma unroll
    for (int c = 0; c < 8; ++c)
        if (c < D) o[c] = acc[c];
}

static int launch_blend_pixel(const BlendParams& p, cudaStream_t st)
{
    const int64_t npix = (int64_t)p.cam.width * p.cam.height;
    blend_pixel_kernel<<<(unsigned)((npix + kPixThreads - 1) / kPixThreads), kPixThreads, 0, st>>>(p);
    QR_LAUNCH_OK("blend_pixel_kernel");
    return QR_OK;
}

}  // namespace qr

extern "C" size_t qr_forward_workspace_bytes(const qr_camera* cam, int32_t K, int32_t D)
{
    (void)D;
    if (!cam || cam->width < 1 || cam->height < 1 || K < 1 || K > QR_MAX_K) return 0;
    return qr::fwd_layout(qr::make_cam(cam), K).total;
}

// batch_n / view_h: 0 for a single view; qr_forward_batch passes the Gaussians per view and the rows per view
static int forward_impl(const qr_camera* cam, int32_t K, int32_t D, qr_dtype feat_dtype, const float* mean2d,
                        const float* conic_opac, const uint32_t* isect_gauss, const int32_t* tile_range,
                        const void* features, float* out_map, int32_t* sel_idx, float* sel_w, int32_t* n_sel,
                        float* resid_TQ, void* ws, size_t ws_bytes, void* stream, int32_t batch_n, int32_t view_h,
                        bool strat = false, float t_min = 0.0f, float z_max = 2.0f)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (K < 1) return fail(QR_ERR_INVALID_ARG, "qr_forward: K = %d < 1 (SPEC.md:215)", K);
    if (K > QR_MAX_K) return fail(QR_ERR_UNSUPPORTED, "qr_forward: K = %d > QR_MAX_K", K);
    if (int rc = check_feat(D, feat_dtype, "qr_forward")) return rc;
    if (!tile_range || !sel_idx || !sel_w || !n_sel || !resid_TQ || !ws)
        return fail(QR_ERR_NULL_POINTER, "qr_forward: NULL output, tile_range or workspace");
    // out_map == NULL: selection only (walk, records, selection lists; no blend) -- the tcgen05 path only
    if (!out_map && !blend_mma_supported(D, feat_dtype))
        return fail(QR_ERR_NULL_POINTER, "qr_forward: out_map is NULL (selection only needs a shape of the tcgen05 path: D %% 32 == 0, or D < 32 with D %% 4 == 0)");
    if (!aligned16(out_map) || !aligned16(features) || !aligned16(conic_opac) || !aligned16(mean2d) || !aligned16(ws))
        return fail(QR_ERR_MISALIGNED, "qr_forward: out_map / features / conic_opac / mean2d / ws must be 16-byte aligned");
    const Cam c = make_cam(cam);
    const FwdLayout L = fwd_layout(c, K);
    const size_t stats_bytes = strat ? (size_t)c.width * c.height * sizeof(float2) : 0;
    if (ws_bytes < L.total + stats_bytes)
        return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_forward: workspace %zu < %zu bytes", ws_bytes, L.total + stats_bytes);
    if (strat && !blend_mma_supported(D, feat_dtype))
        return fail(QR_ERR_UNSUPPORTED, "qr_forward_stratified: shapes of the tcgen05 path only: D %% 32 == 0, or D < 32 with D %% 4 == 0 (D = %d)", D);
    cudaStream_t st = (cudaStream_t)stream;
    const int T = c.tiles_x * c.tiles_y;
    char* w = static_cast<char*>(ws);

    if (blend_mma_supported(D, feat_dtype)) {
        // walk2_kernel -> selection lists -> tcgen05 blend.  isect_gauss may be NULL when M = 0 (every tile range is empty: it
        // is never read), as on the FFMA paths
        if (!mean2d || !conic_opac || !features)
            return fail(QR_ERR_NULL_POINTER, "qr_forward: NULL input");
        WalkParams2 w2;
        w2.cam = c; w2.K = K;
        w2.mean2d = reinterpret_cast<const float2*>(mean2d);
        w2.conic_opac = reinterpret_cast<const float4*>(conic_opac);
        w2.isect = isect_gauss; w2.tile_range = reinterpret_cast<const int2*>(tile_range);
        w2.n_sel = n_sel; w2.resid = resid_TQ; w2.sel_idx = sel_idx; w2.sel_w = sel_w;
        w2.sl = sel_view(L.sel, ws);
        w2.batch_n = batch_n; w2.view_h = view_h;
        if (strat) {
            w2.stats = reinterpret_cast<float2*>(w + L.total);
            w2.t_min = t_min; w2.z_max = z_max;
            if (int rc = launch_walk2_stratified(w2, st)) return rc;
        } else if (int rc = launch_walk2(w2, st)) return rc;
        if (!out_map) return QR_OK;             // selection only: qr_pooled_loss / qr_backward_lists consume the lists
        BlendParams bp;
        bp.cam = c; bp.K = K; bp.D = D; bp.cap = 0; bp.num_tiles = T; bp.tile_ticket = nullptr;
        bp.features = features; bp.gcount = nullptr; bp.ucount = nullptr; bp.rec = nullptr;
        bp.n_sel = n_sel; bp.resid = resid_TQ; bp.out_map = out_map; bp.sel_idx = sel_idx; bp.sel_w = sel_w;
        bp.sl = w2.sl;
        bp.feat_f16 = feat_dtype == QR_F16 ? 1 : 0;
        return launch_blend_mma(bp, st);
    }

    WalkParams wp;
    wp.cam = c; wp.K = K; wp.cap = L.cap;
    wp.mean2d = reinterpret_cast<const float2*>(mean2d);
    wp.conic_opac = reinterpret_cast<const float4*>(conic_opac);
    wp.isect = isect_gauss; wp.tile_range = reinterpret_cast<const int2*>(tile_range);
    wp.n_sel = n_sel; wp.resid = resid_TQ; wp.sel_idx = sel_idx; wp.sel_w = sel_w;
    wp.tile_ticket = reinterpret_cast<int32_t*>(w + L.ticket);
    wp.gcount = reinterpret_cast<int32_t*>(w + L.gcount);
    wp.ucount = reinterpret_cast<int32_t*>(w + L.ucount);
    wp.rec = reinterpret_cast<float*>(w + L.rec);
    wp.batch_n = batch_n; wp.view_h = view_h;
    const size_t smem = kWalkBatch * (16 + 16 + 8 + 4) + (size_t)(K + 1) * 4;
    walk_kernel<<<(unsigned)T, kWalkThreads, smem, st>>>(wp);
    QR_LAUNCH_OK("walk_kernel");

    BlendParams bp;
    bp.cam = c; bp.K = K; bp.D = D; bp.cap = L.cap; bp.num_tiles = T; bp.tile_ticket = wp.tile_ticket;
    bp.features = features; bp.gcount = wp.gcount; bp.ucount = wp.ucount; bp.rec = wp.rec;
    bp.n_sel = n_sel; bp.resid = resid_TQ; bp.out_map = out_map; bp.sel_idx = sel_idx; bp.sel_w = sel_w;
    if (feat_dtype == QR_F16) {
        if ((D + 255) / 256 == 1) return launch_blend_tu<__half, 1, 8>(bp, st);
        return launch_blend_tu<__half, 2, 8>(bp, st);
    }
    if (D % 4 == 0) {
        switch ((D + 127) / 128) {
            case 1: return launch_blend_tu<float, 1, 4>(bp, st);
            case 2: return launch_blend_tu<float, 2, 4>(bp, st);
            case 3: return launch_blend_tu<float, 3, 4>(bp, st);
            default: return launch_blend_tu<float, 4, 4>(bp, st);
        }
    }
    if (D <= 8) return launch_blend_pixel(bp, st);
    switch ((D + 31) / 32) {
        case 1: return launch_blend<float, 1, 1>(bp, st);
        case 2: return launch_blend<float, 2, 1>(bp, st);
        case 3: return launch_blend<float, 3, 1>(bp, st);
        default: return launch_blend<float, 4, 1>(bp, st);
    }
}

extern "C" int qr_forward(const qr_camera* cam, int32_t K, int32_t D, qr_dtype feat_dtype, const float* mean2d,
                          const float* conic_opac, const uint32_t* isect_gauss, const int32_t* tile_range,
                          const void* features, float* out_map, int32_t* sel_idx, float* sel_w, int32_t* n_sel,
                          float* resid_TQ, void* ws, size_t ws_bytes, void* stream)
{
    return forward_impl(cam, K, D, feat_dtype, mean2d, conic_opac, isect_gauss, tile_range, features, out_map, sel_idx, sel_w,
                        n_sel, resid_TQ, ws, ws_bytes, stream, 0, 0);
}

extern "C" int qr_forward_batch(const qr_camera* tall, int32_t B, int64_t N, int32_t K, int32_t D, qr_dtype feat_dtype,
                                const float* mean2d, const float* conic_opac, const uint32_t* isect_gauss,
                                const int32_t* tile_range, const void* features, float* out_map, int32_t* sel_idx,
                                float* sel_w, int32_t* n_sel, float* resid_TQ, void* ws, size_t ws_bytes, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(tall)) return rc;
    if (B < 1 || B > QR_MAX_BATCH) return fail(QR_ERR_INVALID_ARG, "qr_forward_batch: B = %d outside [1, QR_MAX_BATCH]", B);
    if (tall->height % B != 0 || (tall->height / B) % kTile != 0)
        return fail(QR_ERR_INVALID_ARG, "qr_forward_batch: height %d is not B = %d views of a multiple of 16 rows", tall->height, B);
    if (N < 1 || N * (int64_t)B >= (int64_t(1) << 31)) return fail(QR_ERR_INVALID_ARG, "qr_forward_batch: N outside [1, 2^31 / B)");
    return forward_impl(tall, K, D, feat_dtype, mean2d, conic_opac, isect_gauss, tile_range, features, out_map, sel_idx, sel_w,
                        n_sel, resid_TQ, ws, ws_bytes, stream, (int32_t)N, tall->height / B);
}

// Several K in one walk: walk2_multi_kernel fills the selection lists of every K, then one tcgen05
// blend per K renders its map.  Pointer arrays are HOST arrays of nK device pointers.
extern "C" int qr_forward_multik(const qr_camera* cam, int32_t nK, const int32_t* Ks, int32_t D, qr_dtype feat_dtype,
                                 const float* mean2d, const float* conic_opac, const uint32_t* isect_gauss,
                                 const int32_t* tile_range, const void* features, float* const* out_map,
                                 int32_t* const* sel_idx, float* const* sel_w, int32_t* const* n_sel, float* const* resid_TQ,
                                 void* const* ws, const size_t* ws_bytes, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (nK < 1 || nK > QR_MAX_MULTI_K) return fail(QR_ERR_INVALID_ARG, "qr_forward_multik: nK = %d outside [1, QR_MAX_MULTI_K]", nK);
    if (!Ks || !out_map || !sel_idx || !sel_w || !n_sel || !resid_TQ || !ws || !ws_bytes)
        return fail(QR_ERR_NULL_POINTER, "qr_forward_multik: NULL pointer array");
    if (int rc = check_feat(D, feat_dtype, "qr_forward_multik")) return rc;
    if (!blend_mma_supported(D, feat_dtype))
        return fail(QR_ERR_UNSUPPORTED, "qr_forward_multik: shapes of the tcgen05 path only (D %% 32 == 0, or D < 32 with D %% 4 == 0; D = %d)", D);
    if (!tile_range || !mean2d || !conic_opac || !features) return fail(QR_ERR_NULL_POINTER, "qr_forward_multik: NULL input");
    if (!aligned16(features) || !aligned16(conic_opac) || !aligned16(mean2d))
        return fail(QR_ERR_MISALIGNED, "qr_forward_multik: features / conic_opac / mean2d must be 16-byte aligned");
    const Cam c = make_cam(cam);
    WalkParamsMulti wp;
    wp.cam = c; wp.nK = nK;
    wp.mean2d = reinterpret_cast<const float2*>(mean2d);
    wp.conic_opac = reinterpret_cast<const float4*>(conic_opac);
    wp.isect = isect_gauss; wp.tile_range = reinterpret_cast<const int2*>(tile_range);
    for (int j = 0; j < kMaxMultiK; ++j) {
        const int jj = j < nK ? j : 0;                      // unused slots repeat slot 0 (never touched by the kernel)
        const int K = Ks[jj];
        if (K < 1) return fail(QR_ERR_INVALID_ARG, "qr_forward_multik: K[%d] = %d < 1", jj, K);
        if (K > QR_MAX_K) return fail(QR_ERR_UNSUPPORTED, "qr_forward_multik: K[%d] = %d > QR_MAX_K", jj, K);
        if (!sel_idx[jj] || !sel_w[jj] || !n_sel[jj] || !resid_TQ[jj] || !ws[jj])
            return fail(QR_ERR_NULL_POINTER, "qr_forward_multik: NULL output or workspace for K[%d]", jj);
        if (!aligned16(out_map[jj]) || !aligned16(ws[jj])) return fail(QR_ERR_MISALIGNED, "qr_forward_multik: out_map / ws of K[%d]", jj);
        const FwdLayout L = fwd_layout(c, K);
        if (ws_bytes[jj] < L.total)
            return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_forward_multik: workspace of K[%d]: %zu < %zu bytes", jj, ws_bytes[jj], L.total);
        for (int i = 0; i < jj; ++i)
            if (j < nK && ws[i] == ws[jj]) return fail(QR_ERR_INVALID_ARG, "qr_forward_multik: K[%d] and K[%d] share a workspace", i, jj);
        wp.K[j] = K;
        wp.n_sel[j] = n_sel[jj]; wp.resid[j] = resid_TQ[jj]; wp.sel_idx[j] = sel_idx[jj]; wp.sel_w[j] = sel_w[jj];
        wp.sl[j] = sel_view(L.sel, ws[jj]);
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (int rc = launch_walk2_multi(wp, st)) return rc;
    for (int j = 0; j < nK; ++j) {
        if (!out_map[j]) continue;                          // selection only for this K
        BlendParams bp;
        bp.cam = c; bp.K = wp.K[j]; bp.D = D; bp.cap = 0; bp.num_tiles = c.tiles_x * c.tiles_y; bp.tile_ticket = nullptr;
        bp.features = features; bp.gcount = nullptr; bp.ucount = nullptr; bp.rec = nullptr;
        bp.n_sel = wp.n_sel[j]; bp.resid = wp.resid[j]; bp.out_map = out_map[j]; bp.sel_idx = wp.sel_idx[j]; bp.sel_w = wp.sel_w[j];
        bp.sl = wp.sl[j];
        bp.feat_f16 = feat_dtype == QR_F16 ? 1 : 0;
        if (int rc = launch_blend_mma(bp, st, j == 0)) return rc;      // the first blend overlaps the walk's tail (PDL), the others follow
    }
    return QR_OK;
}

extern "C" size_t qr_stratified_workspace_bytes(const qr_camera* cam, int32_t K, int32_t D)
{
    const size_t base = qr_forward_workspace_bytes(cam, K, D);
    if (base == 0) return 0;
    return base + (size_t)cam->width * cam->height * sizeof(float2);
}

extern "C" int qr_forward_stratified(const qr_camera* cam, int32_t K, int32_t D, qr_dtype feat_dtype, float t_min, float z_max,
                                     const float* mean2d, const float* conic_opac, const uint32_t* isect_gauss,
                                     const int32_t* tile_range, const void* features, float* out_map, int32_t* sel_idx,
                                     float* sel_w, int32_t* n_sel, float* resid_TQ, void* ws, size_t ws_bytes, void* stream)
{
    using namespace qr;
    if (!(t_min >= 0.0f)) return fail(QR_ERR_INVALID_ARG, "qr_forward_stratified: t_min must be >= 0");
    if (!(z_max > 0.0f)) return fail(QR_ERR_INVALID_ARG, "qr_forward_stratified: z_max must be > 0");
    return forward_impl(cam, K, D, feat_dtype, mean2d, conic_opac, isect_gauss, tile_range, features, out_map, sel_idx, sel_w,
                        n_sel, resid_TQ, ws, ws_bytes, stream, 0, 0, true, t_min, z_max);
}

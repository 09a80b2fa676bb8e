// qr_forward.cu -- qr_forward: Algorithm 1 for every pixel, then f~^Q = f^Q / (1 - T^Q).
//
// Two kernels, split where the method itself splits ("O(N) transmittance walk" / "O(KC) blend"):
//
// walk_kernel   -- the O(N) part, ALU bound.  CTA = one 16x16 tile, thread = pixel, warp = 16x2 pixels = four
//   4x2-pixel groups.  The tile's depth-sorted list is staged 256 entries at a time in shared memory; each warp
//   first intersects the batch with its own pixel rectangle (lane-parallel box test + ballot), then runs
//   Algorithm 1 lines 3-19 sequentially per pixel over the surviving entries only, in the paper's order and in the
//   fp32 decision arithmetic of DESIGN.md.  A selected Gaussian is not blended here: per 4x2 pixel group the kernel
//   appends one record (Gaussian id, the 8 pixels' weights w^Q, 0 where a pixel did not select it) to the group's
//   list in the workspace -- the group's union of selected Gaussians, in depth order.
//
// blend_kernel  -- the O(KC) part.  CTA = one tile, warp = one pixel group at a time; a lane owns 4 consecutive
//   channels of every 128-channel slab for all 8 pixels (128 fp32 accumulators at D = 512).  For every record of the
//   group's list the feature row is loaded ONCE (128-bit coalesced, one row = one 2 KB burst at D = 512; rows shared
//   by the groups of a tile stay in L1) and applied to the 8 pixels from registers -- 8x fewer row loads than a
//   per-pixel gather, which is what makes the blend FMA bound instead of L1/shared bound.  Epilogue: scale by
//   1/(1 - T^Q) (Algorithm 1 line 20), 128-bit streaming stores of the HWC map; the same warp writes the per-pixel
//   selection records (sel_idx, sel_w, -1/0 padded).
#include "qr_common.cuh"

namespace qr {

constexpr int kWalkThreads = 256;
constexpr int kWalkBatch = 256;
constexpr int kGroupPx = 8;                  // 4x2 pixels
constexpr int kGroupsPerTile = 32;

// workspace layout: tile ticket, gcount[G], rec[G][cap] (G = tiles * 32 groups, cap = 8 K + kSentinels).
// A record is 12 words (48 B, 16-byte aligned): the 8 pixels' weights w^Q, the Gaussian id, 3 words of padding.
// Each list ends with kSentinels records of id -1 / weight 0 so that the blend pipeline can prefetch past the end.
constexpr int kRecWords = 12;
constexpr int kSentinels = 3;
struct FwdLayout {
    size_t ticket, gcount, rec, total;
    int64_t G;
    int cap;
};

static FwdLayout fwd_layout(const Cam& cam, int K)
{
    FwdLayout L;
    L.G = (int64_t)cam.tiles_x * cam.tiles_y * kGroupsPerTile;
    L.cap = kGroupPx * K + kSentinels;
    size_t o = 0;
    L.ticket = o; o = align_up(o + 4, 256);
    L.gcount = o; o = align_up(o + (size_t)L.G * 4, 256);
    L.rec = o;    o = align_up(o + (size_t)L.G * L.cap * kRecWords * 4, 256);
    L.total = o;
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
    int32_t* sel_idx;     // only the padding (slots >= n_sel) is written here
    float* sel_w;
    int32_t* gcount;
    float* rec;
    int32_t* tile_ticket; // blend_kernel's tile queue, reset here
};

__global__ void __launch_bounds__(kWalkThreads) walk_kernel(const WalkParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* ent_co = reinterpret_cast<float4*>(smem_raw);                 // [256] a, b, c, opacity
    float4* ent_box = ent_co + kWalkBatch;                                // [256] x_lo, x_hi, y_lo, y_hi
    float2* ent_xy = reinterpret_cast<float2*>(ent_box + kWalkBatch);     // [256]
    int32_t* ent_id = reinterpret_cast<int32_t*>(ent_xy + kWalkBatch);    // [256]
    float* thr = reinterpret_cast<float*>(ent_id + kWalkBatch);           // [K+1]
    __shared__ int32_t nsel_s[kTile * kTile];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x;
    if (tile == 0 && tid == 0) *p.tile_ticket = 0;
    const int tile_x = tile % p.cam.tiles_x, tile_y = tile / p.cam.tiles_x;
    const int K = p.K;
    // warp = pixel rows 2*warp, 2*warp+1 of the tile; lane -> (x = lane & 15, y = lane >> 4)
    const int px = tile_x * kTile + (lane & 15), py = tile_y * kTile + warp * 2 + (lane >> 4);
    const bool inside = px < p.cam.width && py < p.cam.height;
    const float fpx = (float)px + 0.5f, fpy = (float)py + 0.5f;          // R5
    const float wx_lo = (float)(tile_x * kTile), wx_hi = wx_lo + (float)kTile;
    const float wy_lo = (float)(tile_y * kTile + warp * 2), wy_hi = wy_lo + 2.0f;
    // group of this lane: gx = (lane & 15) >> 2 ; slot of the pixel inside its group q = (lane >> 4) * 4 + (lane & 3)
    const int gx = (lane & 15) >> 2, q = (lane >> 4) * 4 + (lane & 3);
    const uint32_t gbits = (0xFu << (4 * gx)) | (0xFu << (16 + 4 * gx));  // lanes of my group
    const int64_t group = (int64_t)tile * kGroupsPerTile + warp * 4 + gx;
    float* my_rec = p.rec + group * p.cap * kRecWords;

    for (int k = tid; k <= K; k += kWalkThreads)                          // thresholds as printed (R3)
        thr[k] = __fsub_rn(1.0f, __fdiv_rn((float)(k + 1), (float)(K + 1)));
    const float t_break = __fdiv_rn(1.0f, (float)(K + 1));
    const int2 range = p.tile_range[tile];

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
            ent_id[tid] = id; ent_co[tid] = co; ent_xy[tid] = xy; ent_box[tid] = box;
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
                if (sm & gbits) {                       // some pixel of my group selected this Gaussian
                    my_rec[gcnt * kRecWords + q] = wQ;  // 8 lanes write the record's 8 weights (32 contiguous bytes)
                    if (q == 0) my_rec[gcnt * kRecWords + 8] = __int_as_float(ent_id[e]);
                    ++gcnt;
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
    // ---- padding of the selection records (-1 / 0 for slots >= n_sel), coalesced: a tile row is 16*K contiguous
    // words of sel_idx / sel_w.  The used slots are written by blend_kernel (it knows 1/(1 - T^Q) by then). ----
    nsel_s[warp * 32 + lane] = ns;                      // index = (2*warp + (lane>>4))*16 + (lane&15) = y_local*16 + x_local
    __syncthreads();
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

struct BlendParams {
    Cam cam;
    int32_t K, D, cap, num_tiles;
    const void* features;
    const int32_t* gcount;
    const float* rec;
    const int32_t* n_sel;
    const float* resid;
    float* out_map;
    int32_t* sel_idx;
    float* sel_w;
    int32_t* tile_ticket;
};

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
    const int D = p.D, K = p.K;
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

        // lanes 0..7 own the bookkeeping of pixel q = lane: 1/(1 - T^Q) and the record cursor
        const int mx = gx0 + (lane & 3), my = gy0 + ((lane >> 2) & 1);
        const bool mine = lane < kGroupPx && mx < p.cam.width && my < p.cam.height;
        const int64_t mpix = (int64_t)my * p.cam.width + mx;
        const float minv = cur.inv;
        int32_t* my_idx = p.sel_idx + mpix * K;
        float* my_w = p.sel_w + mpix * K;

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
            // selection record of pixel q = lane, in list (= depth) order
            if (mine && m.wm != 0.0f) {
                *my_idx++ = id;
                *my_w++ = __fmul_rn(m.wm, minv);
            }
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

static int sm_count()
{
    static int n = 0;
    if (n == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0)
            n = 148;
    }
    return n;
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

}  // namespace qr

extern "C" size_t qr_forward_workspace_bytes(const qr_camera* cam, int32_t K, int32_t D)
{
    (void)D;
    if (!cam || cam->width < 1 || cam->height < 1 || K < 1 || K > QR_MAX_K) return 0;
    return qr::fwd_layout(qr::make_cam(cam), K).total;
}

extern "C" int qr_forward(const qr_camera* cam, int32_t K, int32_t D, qr_dtype feat_dtype, const float* mean2d,
                          const float* conic_opac, const uint32_t* isect_gauss, const int32_t* tile_range,
                          const void* features, float* out_map, int32_t* sel_idx, float* sel_w, int32_t* n_sel,
                          float* resid_TQ, void* ws, size_t ws_bytes, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (K < 1) return fail(QR_ERR_INVALID_ARG, "qr_forward: K = %d < 1 (SPEC.md:215)", K);
    if (K > QR_MAX_K) return fail(QR_ERR_UNSUPPORTED, "qr_forward: K = %d > QR_MAX_K", K);
    if (int rc = check_feat(D, feat_dtype, "qr_forward")) return rc;
    if (!tile_range || !out_map || !sel_idx || !sel_w || !n_sel || !resid_TQ || !ws)
        return fail(QR_ERR_NULL_POINTER, "qr_forward: NULL output, tile_range or workspace");
    if (!aligned16(out_map) || !aligned16(features) || !aligned16(conic_opac) || !aligned16(mean2d) || !aligned16(ws))
        return fail(QR_ERR_MISALIGNED, "qr_forward: out_map / features / conic_opac / mean2d / ws must be 16-byte aligned");
    const Cam c = make_cam(cam);
    const FwdLayout L = fwd_layout(c, K);
    if (ws_bytes < L.total)
        return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_forward: workspace %zu < %zu bytes", ws_bytes, L.total);
    cudaStream_t st = (cudaStream_t)stream;
    const int T = c.tiles_x * c.tiles_y;
    char* w = static_cast<char*>(ws);

    WalkParams wp;
    wp.cam = c; wp.K = K; wp.cap = L.cap;
    wp.mean2d = reinterpret_cast<const float2*>(mean2d);
    wp.conic_opac = reinterpret_cast<const float4*>(conic_opac);
    wp.isect = isect_gauss; wp.tile_range = reinterpret_cast<const int2*>(tile_range);
    wp.n_sel = n_sel; wp.resid = resid_TQ; wp.sel_idx = sel_idx; wp.sel_w = sel_w;
    wp.tile_ticket = reinterpret_cast<int32_t*>(w + L.ticket);
    wp.gcount = reinterpret_cast<int32_t*>(w + L.gcount);
    wp.rec = reinterpret_cast<float*>(w + L.rec);
    const size_t smem = kWalkBatch * (16 + 16 + 8 + 4) + (size_t)(K + 1) * 4;
    walk_kernel<<<(unsigned)T, kWalkThreads, smem, st>>>(wp);
    QR_LAUNCH_OK("walk_kernel");

    BlendParams bp;
    bp.cam = c; bp.K = K; bp.D = D; bp.cap = L.cap; bp.num_tiles = T; bp.tile_ticket = wp.tile_ticket;
    bp.features = features; bp.gcount = wp.gcount; bp.rec = wp.rec;
    bp.n_sel = n_sel; bp.resid = resid_TQ; bp.out_map = out_map; bp.sel_idx = sel_idx; bp.sel_w = sel_w;
    if (feat_dtype == QR_F16) {
        if ((D + 255) / 256 == 1) return launch_blend<__half, 1, 8>(bp, st);
        return launch_blend<__half, 2, 8>(bp, st);
    }
    if (D % 4 == 0) {
        switch ((D + 127) / 128) {
            case 1: return launch_blend<float, 1, 4>(bp, st);
            case 2: return launch_blend<float, 2, 4>(bp, st);
            case 3: return launch_blend<float, 3, 4>(bp, st);
            default: return launch_blend<float, 4, 4>(bp, st);
        }
    }
    switch ((D + 31) / 32) {
        case 1: return launch_blend<float, 1, 1>(bp, st);
        case 2: return launch_blend<float, 2, 1>(bp, st);
        case 3: return launch_blend<float, 3, 1>(bp, st);
        default: return launch_blend<float, 4, 1>(bp, st);
    }
}

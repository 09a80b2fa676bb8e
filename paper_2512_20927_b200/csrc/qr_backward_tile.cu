// qr_backward_tile.cu -- qr_backward as a persistent, warp-specialised kernel:
//     dL/dF[i,:] += sum_{p, s : sel_idx[p,s] = i}  sel_w[p,s] * dL_dmap[p,:]
//
// Per 16x8-pixel half tile this is  dF_part[U, D] = W^T[U, 128 px] . G[128 px, D]  with U the union of the Gaussians
// selected by any of the 128 pixels (mean 47 at config 3) and W 25-30 % dense.  One CTA per SM, 12 warps:
//   warps 0..7   consumers.  Warp w keeps 8 union rows x all D channels in registers (lane = 4 consecutive channels
//                of every 128-channel slab: 128 fp32 accumulators at D = 512) and streams the unit's pixels: one
//                LDS + ballot finds, for 4 pixels at a time, which of its 8 rows each pixel selected; only then is
//                the pixel's dL_dmap row read from shared memory (128-bit) and applied with packed FFMA2 to exactly
//                the selected rows (warp-uniform branches: no padding work).  Flush: one vector reduction per
//                (union row, 4 channels), so global atomics drop from (sum of n_sel) D to (sum of unions) D.
//   warps 8..10  setup, one unit ahead of the consumers: number the distinct selected Gaussians of the unit with a
//                shared-memory hash set and scatter the weights into the dense block W[px][64 rows] (double buffered).
//                Union slot c goes to consumer warp c % 8, so the 8 warps carry equal numbers of rows.
//   warp  11     loader: one bulk async copy (TMA, mbarrier complete_tx) per 8 pixels of dL_dmap -- 8 consecutive
//                pixels of an image row are 8 D contiguous floats -- into a ring of stages, far ahead of use.
// A unit is (half tile, range of 8-pixel stages, pass): the stage range is cut so that the unit's records fit the
// hash set, and a union larger than 64 rows is processed in passes of 64 rows that re-stream the same pixels.
#include "qr_async.cuh"
#include "qr_backward.cuh"

namespace qr {

using namespace aq;

constexpr int kBtConsumers = 8;
constexpr int kBtSetupWarps = 3;
constexpr int kBtSetupThreads = kBtSetupWarps * 32;
constexpr int kBtThreads = 384;           // warps 0..7 consumers, 8..10 setup, 11 loader; 168 registers per thread
                                          // hold the 128 accumulators, so no setmaxnreg re-split is needed
constexpr int kBtPx = 128;                // half tile: 16 x 8 pixels
constexpr int kBtStagePx = 8;
constexpr int kBtStagesPerUnit = kBtPx / kBtStagePx;   // 16
constexpr int kBtRows = 64;               // union rows per pass
constexpr int kBtSlab = kBtPx * 8;        // W[b][warp][px][8 rows]: words per consumer warp
constexpr int kBtHash = 4096;
constexpr int kBtCap = 3072;              // staged records per unit, each pixel padded to a multiple of 4
                                          // (hash load <= 0.75); 8 px x QR_MAX_K = 2048 always fits

struct BtDesc {
    int32_t ht, j0, j1, nrows, flags;     // flags: 1 = no more work
    int32_t uid[kBtRows];                 // column (w * 8 + r) -> Gaussian id
};

struct BtSmem {
    int ring, W, hkey, hslot, sid, sw, spx, nsel, E, desc, bars, total;
};
__host__ __device__ inline BtSmem bt_smem(int D, int stages)
{
    BtSmem L;
    int o = 0;
    L.ring = o;  o += stages * kBtStagePx * D * 4;
    L.W = o;     o += 2 * kBtConsumers * kBtSlab * 4;
    L.hkey = o;  o += kBtHash * 4;
    L.sid = o;   o += 2 * kBtCap * 4;
    L.sw = o;    o += 2 * kBtCap * 4;
    L.spx = o;   o += 2 * kBtCap;
    L.hslot = o; o += kBtHash * 2;
    L.nsel = o;  o += 3 * kBtPx * 4;
    L.E = o;     o += 3 * (kBtPx + 4) * 4;
    L.desc = o;  o += 2 * (int)sizeof(BtDesc);
    o = (o + 15) & ~15;
    L.bars = o;  o += (2 * stages + 4) * 8;
    L.total = (o + 15) & ~15;
    return L;
}


__device__ __forceinline__ void bt_red4(float* dst, const float2& a, const float2& b)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y) : "memory");
}
__device__ __forceinline__ void bt_cp16(void* dst, const void* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void bt_cp4(void* dst, const void* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(s32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void bt_cp_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

template <int NV, bool FULL>
__global__ void __launch_bounds__(kBtThreads, 1) backward_tile_kernel(const BackwardParams p, const int stages)
{
    extern __shared__ __align__(128) unsigned char smem[];
    const int D = p.D, K = p.K;
    const BtSmem L = bt_smem(D, stages);
    float* ring = reinterpret_cast<float*>(smem + L.ring);
    float* Wbuf = reinterpret_cast<float*>(smem + L.W);
    BtDesc* desc = reinterpret_cast<BtDesc*>(smem + L.desc);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + L.bars);
    uint64_t* empty = full + stages;
    uint64_t* unit_full = empty + stages;       // [2] setup -> consumers, loader
    uint64_t* unit_empty = unit_full + 2;       // [2] consumers (8) + loader (1) -> setup

    if (p.only_flagged && *p.prep_nflag == 0) return;       // nothing was left to this kernel (the usual case)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int num_half = p.cam.tiles_x * p.cam.tiles_y * 2;
    const int stage_floats = kBtStagePx * D;

    if (tid == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], kBtConsumers); }
        for (int b = 0; b < 2; ++b) { mbar_init(&unit_full[b], 1); mbar_init(&unit_empty[b], kBtConsumers + 1); }
        mbar_fence_init();
    }
    __syncthreads();

    if (warp >= kBtConsumers) {
        if (warp == kBtConsumers + kBtSetupWarps) {
            // ================================================ loader ================================================
            if (lane == 0) {
                int s = 0;
                uint32_t ph = 1;
                for (int unit = 0;; ++unit) {
                    const int b = unit & 1;
                    mbar_wait(&unit_full[b], (unit >> 1) & 1);
                    const int ht = desc[b].ht, j0 = desc[b].j0, j1 = desc[b].j1, flags = desc[b].flags;
                    mbar_arrive(&unit_empty[b]);
                    if (flags & 1) break;
                    const int tile = ht >> 1;
                    const int x0 = (tile % p.cam.tiles_x) * kTile, y0 = (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8;
                    for (int j = j0; j < j1; ++j) {
                        mbar_wait(&empty[s], ph);
                        const int x = x0 + (j & 1) * kBtStagePx, y = y0 + (j >> 1);
                        const int npx = y < p.cam.height ? max(0, min(kBtStagePx, p.cam.width - x)) : 0;
                        if (npx > 0) {
                            const uint32_t bytes = (uint32_t)npx * (uint32_t)D * 4u;
                            mbar_arrive_expect_tx(&full[s], bytes);
                            bulk_g2s(ring + (size_t)s * stage_floats, p.dL_dmap + ((int64_t)y * p.cam.width + x) * D, bytes, &full[s]);
                        } else {
                            mbar_arrive(&full[s]);
                        }
                        if (++s == stages) { s = 0; ph ^= 1u; }
                    }
                }
            }
        } else {
            // ================================================ setup =================================================
            // Software pipeline over this CTA's half tiles h_0, h_1, ...: while h_i is hashed and scattered out of
            // shared memory, the selection records of h_(i+1) and the n_sel of h_(i+2) are in flight (cp.async), so
            // no global-load latency sits on the path that feeds the consumers.
            const int st = tid - kBtConsumers * 32;      // 0..95
            int32_t* hkey = reinterpret_cast<int32_t*>(smem + L.hkey);
            uint16_t* hslot = reinterpret_cast<uint16_t*>(smem + L.hslot);
            int32_t* sid_all = reinterpret_cast<int32_t*>(smem + L.sid);
            float* sw_all = reinterpret_cast<float*>(smem + L.sw);
            uint8_t* spx_all = smem + L.spx;
            int32_t* nsel_all = reinterpret_cast<int32_t*>(smem + L.nsel);
            int32_t* E_all = reinterpret_cast<int32_t*>(smem + L.E);
            __shared__ int32_t ucount;
            const bool k4 = (K & 3) == 0;
            auto ssync = [&]() { named_sync<1, kBtSetupThreads>(); };
            auto origin = [&](int ht, int& x0, int& y0) {
                const int tile = ht >> 1;
                x0 = (tile % p.cam.tiles_x) * kTile;
                y0 = (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8;
            };
            auto next_ht = [&](int ht) {                 // next half tile of this CTA that has rows inside the image
                while (true) {
                    ht += gridDim.x;
                    if (ht >= num_half) return num_half;
                    int x0, y0;
                    origin(ht, x0, y0);
                    if (y0 >= p.cam.height) continue;
                    if (p.only_flagged && p.sl.hdr[(size_t)ht * kHdrWords + 5] == 0) continue;   // the tcgen05 kernel did this one
                    return ht;
                }
            };
            // pixel pl of a half tile: stage j = pl >> 3 covers row j >> 1, x = 8 (j & 1) .. + 7
            auto pix_of = [&](int x0, int y0, int pl, int64_t& pix) -> bool {
                const int j = pl >> 3, x = x0 + (j & 1) * kBtStagePx + (pl & 7), y = y0 + (j >> 1);
                pix = (int64_t)y * p.cam.width + x;
                return x < p.cam.width && y < p.cam.height;
            };
            auto issue_nsel = [&](int ht, int nb) {      // n_sel of the 128 pixels -> nsel_all[nb] (async)
                if (ht >= num_half) return;
                int x0, y0;
                origin(ht, x0, y0);
                for (int pl = st; pl < kBtPx; pl += kBtSetupThreads) {
                    int64_t pix;
                    if (pix_of(x0, y0, pl, pix)) bt_cp4(&nsel_all[nb * kBtPx + pl], p.n_sel + pix);
                    else nsel_all[nb * kBtPx + pl] = 0;
                }
            };
            auto plan = [&](int nb) {                    // clamp n_sel, E = exclusive scan of the padded counts
                if (st < 32) {
                    int32_t* ns = nsel_all + nb * kBtPx + st * 4;
                    int v[4], sum = 0;
#pragma unroll
                    for (int k = 0; k < 4; ++k) { v[k] = max(0, min(K, ns[k])); ns[k] = v[k]; sum += (v[k] + 3) & ~3; }
                    int inc = sum;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (st >= o) inc += t; }
                    int e = inc - sum;
                    int32_t* E = E_all + nb * (kBtPx + 4) + st * 4;
#pragma unroll
                    for (int k = 0; k < 4; ++k) { E[k] = e; e += (v[k] + 3) & ~3; }
                    if (st == 31) E_all[nb * (kBtPx + 4) + kBtPx] = e;
                }
                ssync();
            };
            auto range_end = [&](int nb, int j0) {       // as many 8-pixel stages as fit the staging buffers
                const int32_t* E = E_all + nb * (kBtPx + 4);
                int j1 = j0 + 1;
                while (j1 < kBtStagesPerUnit && E[(j1 + 1) * kBtStagePx] - E[j0 * kBtStagePx] <= kBtCap) ++j1;
                return j1;
            };
            auto issue_rec = [&](int ht, int nb, int sb, int j0, int j1) {   // records of stages [j0, j1) -> staging sb
                int x0, y0;
                origin(ht, x0, y0);
                const int32_t* E = E_all + nb * (kBtPx + 4);
                const int base = E[j0 * kBtStagePx];
                int32_t* sid = sid_all + sb * kBtCap;
                float* sw = sw_all + sb * kBtCap;
                uint8_t* spx = spx_all + sb * kBtCap;
                for (int pl = j0 * kBtStagePx + st; pl < j1 * kBtStagePx; pl += kBtSetupThreads) {
                    const int ns = nsel_all[nb * kBtPx + pl];
                    if (ns == 0) continue;
                    int64_t pix;
                    pix_of(x0, y0, pl, pix);
                    const int o = E[pl] - base;
                    const int32_t* gi = p.sel_idx + pix * K;
                    const float* gw = p.sel_w + pix * K;
                    if (k4) {
                        for (int c = 0; c < ns; c += 4) {
                            bt_cp16(sid + o + c, gi + c);
                            bt_cp16(sw + o + c, gw + c);
                            *reinterpret_cast<uint32_t*>(spx + o + c) = (uint32_t)pl * 0x01010101u;
                        }
                    } else {
                        for (int c = 0; c < ns; ++c) {
                            bt_cp4(sid + o + c, gi + c);
                            bt_cp4(sw + o + c, gw + c);
                            spx[o + c] = (uint8_t)pl;
                        }
                    }
                }
            };
            auto fixup = [&](int nb, int sb, int j0, int j1) {   // padding entries of every pixel: id -1
                const int32_t* E = E_all + nb * (kBtPx + 4);
                const int base = E[j0 * kBtStagePx];
                int32_t* sid = sid_all + sb * kBtCap;
                for (int pl = j0 * kBtStagePx + st; pl < j1 * kBtStagePx; pl += kBtSetupThreads) {
                    const int ns = nsel_all[nb * kBtPx + pl];
                    const int o = E[pl] - base;
                    for (int c = ns; c < ((ns + 3) & ~3); ++c) sid[o + c] = -1;
                }
            };

            int unit = 0;
            int ht = blockIdx.x - (int)gridDim.x;
            ht = next_ht(ht);
            int ht1 = ht < num_half ? next_ht(ht) : num_half;
            // prologue: n_sel(h_0) synchronously, records(h_0) and n_sel(h_1) in flight
            issue_nsel(ht, 0);
            bt_cp_wait_all();
            ssync();
            if (ht < num_half) {
                plan(0);
                issue_rec(ht, 0, 0, 0, range_end(0, 0));
                issue_nsel(ht1, 1);
            }
            for (int i = 0; ht < num_half; ++i) {
                const int nb = i % 3, sb = i & 1;
                const int32_t* E = E_all + nb * (kBtPx + 4);
                bt_cp_wait_all();
                ssync();                                 // records(h_i, first range) and n_sel(h_(i+1)) have landed
                const int ht2 = ht1 < num_half ? next_ht(ht1) : num_half;
                if (ht1 < num_half) {
                    const int nb1 = (i + 1) % 3;
                    plan(nb1);
                    issue_rec(ht1, nb1, sb ^ 1, 0, range_end(nb1, 0));
                    issue_nsel(ht2, (i + 2) % 3);
                }
                int j0 = 0;
                while (j0 < kBtStagesPerUnit) {
                    const int j1 = range_end(nb, j0);
                    const int R = E[j1 * kBtStagePx] - E[j0 * kBtStagePx];
                    if (R == 0) { j0 = j1; continue; }                 // nothing selected in these stages: no unit
                    if (j0 > 0) {                                     // later range of the same half tile (rare)
                        ssync();
                        issue_rec(ht, nb, sb, j0, j1);
                        bt_cp_wait_all();
                        ssync();
                    }
                    fixup(nb, sb, j0, j1);
                    int hs = 64;
                    while (hs < 2 * R) hs <<= 1;
                    hs = min(hs, kBtHash);
                    const int hmask = hs - 1;
                    {
                        int4* hz = reinterpret_cast<int4*>(hkey);
                        for (int k = st; k < hs / 4; k += kBtSetupThreads) hz[k] = make_int4(-1, -1, -1, -1);
                    }
                    if (st == 0) ucount = 0;
                    ssync();
                    const int32_t* sid = sid_all + sb * kBtCap;
                    const float* sw = sw_all + sb * kBtCap;
                    const uint8_t* spx = spx_all + sb * kBtCap;
                    // ---- insert the ids; the thread that creates a cell numbers it ----
                    for (int k = st; k < R; k += kBtSetupThreads) {
                        const int32_t id = sid[k];
                        if (id < 0) continue;
                        uint32_t h = hash32((uint32_t)id) & hmask;
                        while (true) {
                            const int32_t old = atomicCAS(&hkey[h], -1, id);
                            if (old == -1) { hslot[h] = (uint16_t)atomicAdd(&ucount, 1); break; }
                            if (old == id) break;
                            h = (h + 1) & hmask;
                        }
                    }
                    ssync();
                    const int U = ucount;
                    const int npass = (U + kBtRows - 1) / kBtRows;
                    for (int pass = 0; pass < npass; ++pass, ++unit) {
                        const int b = unit & 1;
                        mbar_wait(&unit_empty[b], ((unit >> 1) & 1) ^ 1);
                        float* Wb = Wbuf + b * kBtConsumers * kBtSlab;
                        {
                            const int n4 = (j1 - j0) * kBtStagePx * 2;           // float4 per consumer slab
                            for (int k = st; k < n4 * kBtConsumers; k += kBtSetupThreads) {
                                const int w = k / n4, r = k - w * n4;
                                reinterpret_cast<float4*>(Wb + w * kBtSlab + j0 * kBtStagePx * 8)[r] = make_float4(0.f, 0.f, 0.f, 0.f);
                            }
                        }
                        ssync();
                        for (int k = st; k < R; k += kBtSetupThreads) {
                            const int32_t id = sid[k];
                            if (id < 0) continue;
                            uint32_t h = hash32((uint32_t)id) & hmask;
                            while (hkey[h] != id) h = (h + 1) & hmask;
                            const int c = (int)hslot[h] - pass * kBtRows;
                            if (c >= 0 && c < kBtRows) {
                                const int cw = c & 7, r = c >> 3;                  // consumer warp c % 8, its row c / 8
                                Wb[cw * kBtSlab + (int)spx[k] * 8 + r] = sw[k];
                                desc[b].uid[cw * 8 + r] = id;
                            }
                        }
                        if (st == 0) {
                            desc[b].ht = ht; desc[b].j0 = j0; desc[b].j1 = j1; desc[b].flags = 0;
                            desc[b].nrows = min(kBtRows, U - pass * kBtRows);
                        }
                        __threadfence_block();
                        ssync();
                        if (st == 0) mbar_arrive(&unit_full[b]);
                    }
                    j0 = j1;
                }
                ht = ht1; ht1 = ht2;
            }
            {
                const int b = unit & 1;
                mbar_wait(&unit_empty[b], ((unit >> 1) & 1) ^ 1);
                if (st == 0) { desc[b].flags = 1; desc[b].j0 = desc[b].j1 = 0; __threadfence_block(); mbar_arrive(&unit_full[b]); }
            }
        }
    } else {
        // ================================================== consumers ===============================================
        float2 acc[8][NV][2];
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int j = 0; j < NV; ++j) acc[r][j][0] = acc[r][j][1] = make_float2(0.f, 0.f);
        int s = 0;
        uint32_t ph = 0;
        for (int unit = 0;; ++unit) {
            const int b = unit & 1;
            mbar_wait(&unit_full[b], (unit >> 1) & 1);
            const BtDesc* d = &desc[b];
            if (d->flags & 1) break;
            const int j0 = d->j0, j1 = d->j1, nrows = d->nrows;
            const float* Ws = Wbuf + (b * kBtConsumers + warp) * kBtSlab;      // this warp's [px][8 rows]
            for (int j = j0; j < j1; ++j) {
                mbar_wait(&full[s], ph);
                const float* gs = ring + (size_t)s * stage_floats + lane * 4;
#pragma unroll
                for (int hq = 0; hq < 2; ++hq) {
                    // lane = (pixel hq*4 + (lane >> 3) of the stage, row lane & 7 of this warp)
                    const float* Wp = Ws + (j * kBtStagePx + hq * 4) * 8;
                    const uint32_t m32 = __ballot_sync(0xffffffffu, Wp[lane] != 0.0f);
                    if (m32 == 0u) continue;
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const uint32_t m = (m32 >> (8 * q)) & 0xFFu;
                        if (m == 0u) continue;
                        const float* gp = gs + (hq * 4 + q) * D;
                        float4 g[NV];
#pragma unroll
                        for (int jj = 0; jj < NV; ++jj) {
                            if (FULL || (jj * 32 + lane) * 4 < D) g[jj] = *reinterpret_cast<const float4*>(gp + jj * 128);
                            else g[jj] = make_float4(0.f, 0.f, 0.f, 0.f);
                        }
                        const float4 wa = *reinterpret_cast<const float4*>(Wp + q * 8);
                        const float4 wb = *reinterpret_cast<const float4*>(Wp + q * 8 + 4);
                        const float w8[8] = { wa.x, wa.y, wa.z, wa.w, wb.x, wb.y, wb.z, wb.w };
#pragma unroll
                        for (int r = 0; r < 8; ++r) {
                            if (m & (1u << r)) {
                                const float2 ww = make_float2(w8[r], w8[r]);
#pragma unroll
                                for (int jj = 0; jj < NV; ++jj) {
                                    acc[r][jj][0] = __ffma2_rn(ww, make_float2(g[jj].x, g[jj].y), acc[r][jj][0]);
                                    acc[r][jj][1] = __ffma2_rn(ww, make_float2(g[jj].z, g[jj].w), acc[r][jj][1]);
                                }
                            }
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[s]);
                if (++s == stages) { s = 0; ph ^= 1u; }
            }
            // ---- flush: one vector reduction per (union row, 4 channels) ----
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                if (r * 8 + warp < nrows) {
                    float* drow = p.dL_dfeat + (int64_t)d->uid[warp * 8 + r] * D + lane * 4;
#pragma unroll
                    for (int jj = 0; jj < NV; ++jj) {
                        if (FULL || (jj * 32 + lane) * 4 < D) bt_red4(drow + jj * 128, acc[r][jj][0], acc[r][jj][1]);
                        acc[r][jj][0] = acc[r][jj][1] = make_float2(0.f, 0.f);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&unit_empty[b]);
        }
    }
}

bool backward_tile_supported(int32_t K, int32_t D) { return D % 4 == 0 && D >= 4 && D <= 512 && K >= 1 && K <= QR_MAX_K; }

template <int NV>
static int launch_bt(const BackwardParams& p, cudaStream_t st)
{
    const int sms = sm_count();
    const int num_half = p.cam.tiles_x * p.cam.tiles_y * 2;
    const unsigned grid = (unsigned)min(sms, num_half);
    const int stages = max(2, min(12, (80 * 1024) / (kBtStagePx * p.D * 4)));   // ring <= 80 KB next to 146 KB of setup state
    const int smem = bt_smem(p.D, stages).total;
    if (p.D == NV * 128) {
        auto kern = backward_tile_kernel<NV, true>;
        QR_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        kern<<<grid, kBtThreads, smem, st>>>(p, stages);
    } else {
        auto kern = backward_tile_kernel<NV, false>;
        QR_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        kern<<<grid, kBtThreads, smem, st>>>(p, stages);
    }
    QR_LAUNCH_OK("backward_tile_kernel");
    return QR_OK;
}

int launch_backward_tile(const BackwardParams& p, cudaStream_t st)
{
    switch ((p.D + 127) / 128) {
        case 1: return launch_bt<1>(p, st);
        case 2: return launch_bt<2>(p, st);
        case 3: return launch_bt<3>(p, st);
        default: return launch_bt<4>(p, st);
    }
}

}  // namespace qr

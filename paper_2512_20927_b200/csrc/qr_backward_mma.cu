// qr_backward_mma.cu -- qr_backward as a dense contraction on the 5th-generation
// tensor cores:
//     dL/dF[i,:] += sum_{p, s : sel_idx[p,s] = i}  sel_w[p,s] * dL_dmap[p,:]
//
// Per 16x8-pixel half tile this is  dF_part^T[D, U] = G^T[D, 128 px] . W[128 px, U]  with U the union of the Gaussians
// selected by any of the 128 pixels (mean 47 at config 3) and W the sparse weights.  ncu showed the FFMA formulation
// (qr_backward_tile.cu) to be latency / issue bound at 4x the time of its HBM traffic (profiles/README.md, r1_b): only
// 16 % of its warp instructions are FFMA2, the rest finds out which of a warp's rows a pixel selected.  On the tensor
// core the zero weights cost nothing extra and the operands never pass through registers.
//
// Shape: M = 128 channels (TMEM lane = channel), N = 64 union rows, K = 8 pixels per tcgen05.mma (kind::tf32).
//   A = G^T, "MN-major": dL_dmap is [pixel][channel] with channels contiguous.  One TMA tensor copy per 32 channels
//       (box = 32 channels x 8 consecutive pixels of an image row, SWIZZLE_128B_ATOM_32B) lands a stage directly in
//       the layout the MMA reads (UMMA SWIZZLE_128B_BASE32B): no thread ever moves dL_dmap.
//   B = W, K-major, no swizzle: scattered by the setup warps from the entry lists backward_prep_kernel wrote.
// Precision: kind::tf32 truncates fp32 operands to 10 explicit mantissa bits (measured on B200), so the raw G tile IS
// G_hi; converter warps write G_lo = G - trunc(G) next to it, W is split exactly into W_hi + W_lo, and three MMAs
// accumulate G_hi W_hi + G_hi W_lo + G_lo W_hi in fp32 (TMEM).  The dropped G_lo W_lo term and the truncation of the
// lo parts are <= 2^-21 relative per product, 40x below the fp32 tolerance of north_star (1e-4 relative).
//
// backward_prep_kernel (one CTA per half tile, high occupancy) numbers the distinct selected Gaussians of every half
// tile and rewrites its selection as pixel-ordered entries {weight, union row << 8 | pixel}: the irregular,
// latency-bound part of the job.  backward_mma_kernel is one persistent CTA per SM, 18 warps, roles by warp (no role
// ever waits at a block barrier):
//   warps 0..3    epilogue: tcgen05.ld of the accumulator (lane = channel, column = union row), one coalesced
//                 red.global.add.f32 per (union row, 32 channels)
//   warp  4       MMA issue: warp-uniform loop, one elected lane issues tcgen05.mma / tcgen05.commit
//   warp  5       loader: TMA tensor copies of dL_dmap into a ring of stages, far ahead of use
//   warps 6..13   converters: G_lo = G - trunc(G), elementwise over a stage (same swizzled offset in the lo ring)
//   warps 14..17  setup, one unit ahead: stream the unit's entries, clear W and scatter hi / lo.  W is double buffered
//                 by halves of the K range (pixels 0..63 / 64..127): half h of the next unit is rebuilt as soon as
//                 the MMAs that read it have retired.
// A unit is (half tile, pass): a union larger than 64 rows is processed in passes of 64 rows that re-stream the same
// pixels.  Half tiles with more than kBmEntCap records are left to backward_tile_kernel (qr_backward_tile.cu).
#include <cuda.h>

#include "qr_backward.cuh"
#include "qr_umma.cuh"

namespace qr {

using namespace aq;

constexpr int kBmEpiWarps = 4;
constexpr int kBmMmaWarp = 4;
constexpr int kBmLoadWarp = 5;
constexpr int kBmFirstConv = 6;
constexpr int kBmConvWarps = 8;
constexpr int kBmFirstSetup = kBmFirstConv + kBmConvWarps;       // 14
constexpr int kBmSetupWarps = 4;
constexpr int kBmSetupThreads = kBmSetupWarps * 32;
constexpr int kBmThreads = (kBmFirstSetup + kBmSetupWarps) * 32;  // 576
constexpr int kBmPx = 128;                 // half tile: 16 x 8 pixels
constexpr int kBmStagePx = 8;              // one tf32 K step
constexpr int kBmStagesPerUnit = kBmPx / kBmStagePx;   // 16
constexpr int kBmRows = 64;                // union rows per pass = MMA N
constexpr int kBmHalfPx = 64;              // pixels per W half buffer
constexpr int kBmWHalfBytes = kBmRows * kBmHalfPx * 4;           // 16 KB (hi or lo of one half)
constexpr int kBmHash = 8192;              // backward_prep_kernel: hash cells per half tile
constexpr int kBmEntCap = 5120;            // selection records (and distinct Gaussians) of a half tile the tcgen05 path
                                           // takes; fuller half tiles are left to backward_tile_kernel
constexpr int kBmEntRegs = 8;              // entries a setup thread holds in flight
#ifndef KBM_LO
#define KBM_LO 2
#endif
constexpr int kBmLoStages = KBM_LO;             // G_lo is produced just ahead of the MMA that reads it
constexpr int kBmDescRing = 4;

struct BmDesc {
    int32_t ht, j0, j1, nrows, flags, pad; // flags: 1 = no more work
    int64_t row[kBmRows];                  // union row (MMA column) -> offset of the Gaussian's row in dL_dfeat (floats)
};

struct BmSmem {
    int W, stages, desc, bars, misc, total;
};
__host__ __device__ inline int bm_pad(int D) { return (D + 127) & ~127; }
__host__ __device__ inline BmSmem bm_smem(int D, int stages)
{
    BmSmem L;
    int o = 0;
    L.W = o;      o += 2 * 2 * kBmWHalfBytes;                    // [half][hi, lo]
    L.stages = o; o += (stages + kBmLoStages) * kBmStagePx * D * 4;   // [stages] G (= G_hi), then [kBmLoStages] G_lo; 1 KB aligned
    L.desc = o;   o += kBmDescRing * (int)sizeof(BmDesc);
    o = (o + 15) & ~15;
    L.bars = o;   o += (2 * stages + 2 * kBmLoStages + 8) * 8;
    L.misc = o;   o += 16;                                       // TMEM base, done flag, two half-tile ticket slots
    L.total = (o + 15) & ~15;
    return L;
}

__device__ __forceinline__ void bm_cp16(void* dst, const void* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void bm_cp4(void* dst, const void* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(s32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void bm_cp_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
// byte offset of W[row c][pixel k] inside a 16 KB half buffer: K-major, no swizzle; core matrix = 8 rows x 4 pixels
// (128 B); pixel chunks 128 B apart (LBO), 8-row groups 2 KB apart (SBO)
__device__ __forceinline__ uint32_t bm_w_off(int c, int k)
{
    return (uint32_t)((c >> 3) * (kBmHalfPx / 4 * 128) + (k >> 2) * 128 + (c & 7) * 16 + (k & 3) * 4);
}
__device__ __forceinline__ void bm_tma_box(void* dst, const CUtensorMap* map, int c0, int x, int y, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(s32(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(s32(bar)), "r"(c0), "r"(x), "r"(y) : "memory");
}
__device__ __forceinline__ void bm_tma_box4(void* dst, const CUtensorMap* map, int c0, int x, int g, int y, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
                 ::"r"(s32(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(s32(bar)), "r"(c0), "r"(x), "r"(g), "r"(y) : "memory");
}
__device__ __forceinline__ void bm_red(float* dst, float v)
{
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(dst), "f"(v) : "memory");
}

// QR_PROF builds: cycles every role spends waiting on each barrier class, summed over the CTAs into ctrl[16..27] (in
// units of 1,024 cycles; [27] = the CTAs' lifetimes); profiles/README.md, experiment 13
#ifdef QR_PROF
#define BPW(cls, bar, par) do { const long long t_ = clock64(); mbar_wait(bar, par); bpw[cls] += clock64() - t_; } while (0)
#else
#define BPW(cls, bar, par) mbar_wait(bar, par)
#endif
__global__ void __launch_bounds__(kBmThreads, 1)
backward_mma_kernel(const BackwardParams p, const int stages, const __grid_constant__ CUtensorMap g_tmap)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    // D: the channel count the contraction runs on = p.D rounded up to whole 128-channel tiles (the TMA load fills channels
    // beyond p.D with zeros, the epilogue does not write them); p.D itself only sizes the rows of dL_dfeat
    const int D = bm_pad(p.D);
    const BmSmem L = bm_smem(D, stages);
    const int nchunks = D >> 7;                      // 128-channel MMA tiles
    const int stage_half = kBmStagePx * D * 4;       // bytes of a stage's hi (or lo) part
    unsigned char* Wsm = smem + L.W;
    unsigned char* stage_base = smem + L.stages;                          // G stages (the MMA reads them as G_hi)
    unsigned char* lo_base = stage_base + (size_t)stages * stage_half;    // G_lo stages
    BmDesc* desc = reinterpret_cast<BmDesc*>(smem + L.desc);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bars);
    uint64_t* raw_full = bars;                       // [stages] loader (TMA complete_tx) -> converters
    uint64_t* stage_empty = raw_full + stages;       // [stages] MMA (tcgen05.commit) -> loader
    uint64_t* lo_ready = stage_empty + stages;       // [kBmLoStages] converters (4 warp arrivals) -> MMA
    uint64_t* lo_empty = lo_ready + kBmLoStages;     // [kBmLoStages] MMA (tcgen05.commit) -> converters
    uint64_t* w_ready = lo_empty + kBmLoStages;      // [2] setup -> MMA, loader (half 0 also publishes the descriptor)
    uint64_t* w_free = w_ready + 2;                  // [2] MMA (tcgen05.commit) -> setup
    uint64_t* tmem_full = w_free + 2;                // [2] MMA (tcgen05.commit) -> epilogue
    uint64_t* tmem_empty = tmem_full + 2;            // [2] epilogue (4 warp arrivals) -> MMA
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L.misc);
    volatile uint32_t* done_flag = reinterpret_cast<volatile uint32_t*>(smem + L.misc + 4);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int num_half = p.cam.tiles_x * p.cam.tiles_y * 2;
#ifdef QR_PROF
    const long long t_start = clock64();
    long long bpw[11] = { 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0 };
#endif
    if (!sel_stamp_ok(p.sl.stamp, p.cam, p.K)) return;      // not the lists of this camera / K: touch nothing

    if (tid == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(&raw_full[s], 1); mbar_init(&stage_empty[s], 1); }
        for (int s = 0; s < kBmLoStages; ++s) { mbar_init(&lo_ready[s], kBmConvWarps); mbar_init(&lo_empty[s], 1); }
        for (int b = 0; b < 2; ++b) {
            mbar_init(&w_ready[b], 1); mbar_init(&w_free[b], 1);
            mbar_init(&tmem_full[b], 1); mbar_init(&tmem_empty[b], kBmEpiWarps);
        }
        *done_flag = 0u;
        mbar_fence_init();
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(s32(tmem_slot)), "r"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp < kBmEpiWarps) {
        // ================================================= epilogue =================================================
        // thread = channel 32 warp + lane of every 128-channel tile (TMEM lane), columns = union rows of the unit
        auto ld16 = [&](uint32_t taddr, uint32_t (&r)[16]) {
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                         : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                           "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                         : "r"(taddr));
        };
        float* dcol = p.dL_dfeat + warp * 32 + lane;
        const bool lastok = (nchunks - 1) * 128 + warp * 32 + lane < p.D;      // the last 128-channel tile may be partial
        for (int unit = 0;; ++unit) {
            const int buf = unit & 1;
            BPW(0, &tmem_full[buf], (unit >> 1) & 1);
            tc_fence_after();
            const BmDesc* d = &desc[unit % kBmDescRing];
            if (d->flags & 1) break;
            const int nrows = d->nrows;
            const int64_t* row = d->row;
            const uint32_t t0 = tmem_base + ((uint32_t)(warp * 32) << 16) + (uint32_t)(buf * 256);
            // 16 union rows at a time, all channel tiles of them: a row's offset is read once and serves up to four
            // reductions 128 channels apart
#pragma unroll 1
            for (int c0 = 0; c0 < nrows; c0 += 16) {
                uint32_t r0[16], r1[16], r2[16], r3[16];
                ld16(t0 + c0, r0);
                if (nchunks > 1) ld16(t0 + kBmRows + c0, r1);
                if (nchunks > 2) ld16(t0 + 2 * kBmRows + c0, r2);
                if (nchunks > 3) ld16(t0 + 3 * kBmRows + c0, r3);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                if (c0 + 16 >= nrows) {                 // every tcgen05.ld of this accumulator has completed
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&tmem_empty[buf]);
                }
#pragma unroll
                for (int c = 0; c < 16; ++c) {
                    if (c0 + c < nrows && row[c0 + c] >= 0) {
                        float* a = dcol + row[c0 + c];
                        if (nchunks > 1 || lastok) bm_red(a, __uint_as_float(r0[c]));
                        if (nchunks > 1 && (nchunks > 2 || lastok)) bm_red(a + 128, __uint_as_float(r1[c]));
                        if (nchunks > 2 && (nchunks > 3 || lastok)) bm_red(a + 256, __uint_as_float(r2[c]));
                        if (nchunks > 3 && lastok) bm_red(a + 384, __uint_as_float(r3[c]));
                    }
                }
            }
        }
    } else if (warp == kBmMmaWarp) {
        // ================================================= MMA issuer ===============================================
        // M = 128 channels, N = 64 rows, fp32 accumulate, A and B tf32, A MN-major, B K-major
        // N = the unit's union rows rounded up to 16: the tensor core's time per MMA grows with N
        const uint32_t idesc0 = (1u << 4) | (2u << 7) | (2u << 10) | (1u << 15) | ((uint32_t)(128 >> 4) << 24);
        const uint32_t w0 = s32(Wsm), st0 = s32(stage_base), lo0 = s32(lo_base);
        int st = 0, s = 0;                               // st counts stages; s = st % stages without the division
        for (int unit = 0;; ++unit) {
            const int buf = unit & 1;
            BPW(1, &w_ready[0], unit & 1);
            const BmDesc* d = &desc[unit % kBmDescRing];
            const int j0 = d->j0, j1 = d->j1, flags = d->flags;
            const uint32_t idesc = idesc0 | ((uint32_t)(max(16, (d->nrows + 15) & ~15) >> 3) << 17);
            BPW(2, &tmem_empty[buf], ((unit >> 1) & 1) ^ 1);
            tc_fence_after();
            if (flags & 1) {
                if (elect_one()) umma_commit(&tmem_full[buf]);
                break;
            }
            bool have_w1 = false;
            for (int j = j0; j < j1; ++j, ++st) {
                const int h = j >> 3;
                if (h == 1 && !have_w1) { BPW(3, &w_ready[1], unit & 1); have_w1 = true; }
                const int l = st % kBmLoStages;
                BPW(4, &lo_ready[l], (st / kBmLoStages) & 1);      // implies raw_full[s]
                tc_fence_after();
                const uint32_t a_hi = st0 + s * stage_half, a_lo = lo0 + l * stage_half;
                const uint32_t b_hi = w0 + h * 2 * kBmWHalfBytes + (j & 7) * 256, b_lo = b_hi + kBmWHalfBytes;
                const uint64_t db_hi = umma_desc(b_hi, 128, kBmHalfPx / 4 * 128, 0);
                const uint64_t db_lo = umma_desc(b_lo, 128, kBmHalfPx / 4 * 128, 0);
                const uint64_t da_hi0 = umma_desc(a_hi, 1024, 512, 1), da_lo0 = umma_desc(a_lo, 1024, 512, 1);
                const uint32_t d0 = tmem_base + (uint32_t)(buf * 256);
#ifdef QR_PROF
                const long long t_issue = clock64();
#endif
                if (elect_one()) {
#pragma unroll 4
                    for (int m = 0; m < nchunks; ++m) {
                        const uint64_t da_hi = da_hi0 + (uint64_t)(m * (4096 >> 4)), da_lo = da_lo0 + (uint64_t)(m * (4096 >> 4));
                        const uint32_t d_tmem = d0 + (uint32_t)(m * kBmRows);
                        umma_tf32(d_tmem, da_hi, db_hi, idesc, j != j0);
                        umma_tf32(d_tmem, da_hi, db_lo, idesc, true);
                        umma_tf32(d_tmem, da_lo, db_hi, idesc, true);
                    }
                    umma_commit(&stage_empty[s]);
                    umma_commit(&lo_empty[l]);
                    if (h == 0 && (j == 7 || j == j1 - 1)) umma_commit(&w_free[0]);     // last read of W half 0
                }
                __syncwarp();
#ifdef QR_PROF
                bpw[10] += clock64() - t_issue;           // issuing the stage's MMAs and commits
#endif
                if (++s == stages) s = 0;
            }
            if (!have_w1) mbar_wait(&w_ready[1], unit & 1);       // keep the phases of every unit in step
            if (elect_one()) {
                if (j0 >= 8) umma_commit(&w_free[0]);
                umma_commit(&w_free[1]);
                umma_commit(&tmem_full[buf]);
            }
            __syncwarp();
        }
    } else if (warp == kBmLoadWarp) {
        // ================================================= loader ===================================================
        // a stage is D / 32 blocks of [8 px][128 B] (32 channels, swizzled), one behind the other.  The tensor map has the
        // 32-channel group as a dimension of its own BEHIND the pixel dimension, so ONE box {32 ch, 8 px, D / 32 groups, 1 row}
        // lands in exactly that layout: one TMA instruction per stage (issued per 1 KB block, the warp's loop over the lanes'
        // boxes kept the loader busy 95 % of the kernel; profiles/README.md, experiment 13)
        int s = 0;
        uint32_t ph = 1;                                 // parity to wait for on stage_empty[s]
        for (int unit = 0;; ++unit) {
            mbar_wait(&w_ready[0], unit & 1);
            const BmDesc* d = &desc[unit % kBmDescRing];
            const int ht = d->ht, j0 = d->j0, j1 = d->j1, flags = d->flags;
            if (flags & 1) {
                mbar_wait(&stage_empty[s], ph);
                if (lane == 0) { *done_flag = 1u; mbar_arrive(&raw_full[s]); }     // wakes the converters up to stop
                break;
            }
            const int tile = ht >> 1;
            const int x0 = (tile % p.cam.tiles_x) * kTile, y0 = (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8;
            for (int j = j0; j < j1; ++j) {
                BPW(5, &stage_empty[s], ph);
                if (lane == 0) {
                    mbar_arrive_expect_tx(&raw_full[s], (uint32_t)stage_half);
                    bm_tma_box4(stage_base + (size_t)s * stage_half, &g_tmap, 0, x0 + (j & 1) * kBmStagePx, 0, y0 + (j >> 1), &raw_full[s]);
                }
                __syncwarp();
                if (++s == stages) { s = 0; ph ^= 1u; }
            }
        }
    } else if (warp < kBmFirstSetup) {
        // ================================================= converters ===============================================
        // a stage is 2 D float4 = D / 128 per thread; the swizzled offset is the same in the G and the G_lo buffer
        const int ct = tid - kBmFirstConv * 32;              // 0..255
        int s = 0;
        uint32_t ph = 0;                                     // parity to wait for on raw_full[s]
        for (int st = 0;; ++st) {
            const int l = st % kBmLoStages;
            BPW(6, &raw_full[s], ph);
            if (*done_flag) break;
            const float4* hi = reinterpret_cast<const float4*>(stage_base + (size_t)s * stage_half) + ct;
            float4* lo = reinterpret_cast<float4*>(lo_base + (size_t)l * stage_half) + ct;
            float4 v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (u < nchunks) v[u] = hi[u * kBmConvWarps * 32];
            BPW(7, &lo_empty[l], ((st / kBmLoStages) & 1) ^ 1);       // the MMAs that read this G_lo buffer have retired
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (u < nchunks)
                    lo[u * kBmConvWarps * 32] = make_float4(__fsub_rn(v[u].x, tf32_hi(v[u].x)), __fsub_rn(v[u].y, tf32_hi(v[u].y)),
                                                           __fsub_rn(v[u].z, tf32_hi(v[u].z)), __fsub_rn(v[u].w, tf32_hi(v[u].w)));
            fence_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(&lo_ready[l]);
            if (++s == stages) { s = 0; ph ^= 1u; }
        }
    } else {
        // ================================================= setup ====================================================
        // backward_prep_kernel has numbered every half tile's selected Gaussians and left its selection as a compact
        // list of (weight, union row, pixel) entries ordered by pixel.  What remains here is streaming: read the next
        // unit's entries (one coalesced 8-byte load each, issued before the wait on the W half they go to), clear the
        // half, scatter hi / lo, publish.
        const int st = tid - kBmFirstSetup * 32;          // 0..127
        auto ssync_setup = [&]() { named_sync<1, kBmSetupThreads>(); };
        int unit = 0;
        auto inside = [&](int ht) {
            const int tile = ht >> 1;
            return (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8 < p.cam.height;
        };
        struct Hd { int n[4], U, flag; };
        auto load_hd = [&](int ht) -> Hd {
            Hd t;
            t.n[0] = t.n[1] = t.n[2] = t.n[3] = 0; t.U = 0; t.flag = 0;
            if (ht < num_half && inside(ht)) {
                const int32_t* hd = p.sl.hdr + (size_t)ht * kHdrWords;
                const int4 v = __ldg(reinterpret_cast<const int4*>(hd));
                const int2 w = __ldg(reinterpret_cast<const int2*>(hd + 4));
                t.n[0] = v.x; t.n[1] = v.y; t.n[2] = v.z; t.n[3] = v.w; t.U = w.x; t.flag = w.y;
            }
            return t;
        };
        // half tiles are handed out by a global ticket (their cost varies with the union size: a static stride left the
        // slowest CTA ~8 % behind the mean); the ticket after next is requested one half tile early and passed to the other
        // setup threads through two alternating shared-memory slots
        volatile int32_t* tslot = reinterpret_cast<volatile int32_t*>(smem + L.misc + 8);
        int32_t* ticket = p.ticket;
        if (st == 0) { tslot[0] = atomicAdd(ticket, 1); tslot[1] = atomicAdd(ticket, 1); }
        ssync_setup();
        int ht = tslot[0], ht1 = tslot[1];
        ssync_setup();
        Hd cnt = load_hd(ht);
        for (int it = 0; ht < num_half; ++it) {
            const Hd cnt1 = load_hd(ht1);
            if (st == 0) tslot[it & 1] = atomicAdd(ticket, 1);
            const int U = cnt.U;
            const int R = cnt.n[0] + cnt.n[1] + cnt.n[2] + cnt.n[3];
            if (R > 0 && cnt.flag == 0) {                 // flag: left to backward_tile_kernel (too many records for the prep)
                const uint2* ent = p.sl.ent + (size_t)ht * kSelLists * p.sl.qcap;
                const int32_t* uid = p.sl.uid + (size_t)ht * p.sl.ucap;
                const int npass = (U + kBmRows - 1) / kBmRows;
                for (int pass = 0; pass < npass; ++pass, ++unit) {
                    BmDesc* d = &desc[unit % kBmDescRing];
                    const int c_lo = pass * kBmRows;
                    for (int h = 0; h < 2; ++h) {
                        // W half h = pixels 64 h .. 64 h + 63 = lists 2 h and 2 h + 1, read as one flat sequence
                        const int na = cnt.n[2 * h], n = na + cnt.n[2 * h + 1];
                        const uint2* la = ent + (size_t)(2 * h) * p.sl.qcap;
                        const uint2* lb = la + p.sl.qcap;
                        unsigned char* whi = Wsm + h * 2 * kBmWHalfBytes;
                        uint2 e[kBmEntRegs];
                        int64_t rowoff = 0;
                        for (int base = 0; base == 0 || base < n; base += kBmEntRegs * kBmSetupThreads) {
#pragma unroll
                            for (int u = 0; u < kBmEntRegs; ++u) {
                                const int k = base + u * kBmSetupThreads + st;
                                e[u] = k < n ? __ldg(k < na ? la + k : lb + (k - na)) : make_uint2(0u, 0xFFFFFFFFu);
                            }
                            if (base == 0) {
                                if (h == 0 && st < kBmRows && c_lo + st < U) {
                                    const int32_t id = __ldg(uid + c_lo + st);
                                    rowoff = (uint32_t)id < (uint32_t)p.N ? (int64_t)id * p.D : -1;   // never add outside the table
                                }
                                BPW(8, &w_free[h], (unit & 1) ^ 1);      // the MMAs of the previous unit have read this half
                                float4* wz = reinterpret_cast<float4*>(whi);
                                for (int k = st; k < 2 * kBmWHalfBytes / 16; k += kBmSetupThreads) wz[k] = make_float4(0.f, 0.f, 0.f, 0.f);
                                ssync_setup();
                            }
#pragma unroll
                            for (int u = 0; u < kBmEntRegs; ++u) {
                                const int c = sel_col(e[u].y) - c_lo;
                                if (c >= 0 && c < kBmRows) {          // padding entries have column 2^17 - 1
                                    const uint32_t off = bm_w_off(c, sel_pixel(e[u].y) & (kBmHalfPx - 1));
                                    const float w = __uint_as_float(e[u].x), hi = tf32_hi(w);
                                    *reinterpret_cast<float*>(whi + off) = hi;
                                    *reinterpret_cast<float*>(whi + kBmWHalfBytes + off) = __fsub_rn(w, hi);
                                }
                            }
                        }
                        if (h == 0) {
                            if (st < kBmRows) d->row[st] = rowoff;
                            if (st == 0) { d->ht = ht; d->j0 = 0; d->j1 = kBmStagesPerUnit; d->flags = 0; d->nrows = min(kBmRows, U - c_lo); }
                        }
                        fence_async_smem();                            // W is read by the tensor core (async proxy)
                        __threadfence_block();
                        ssync_setup();
                        if (st == 0) mbar_arrive(&w_ready[h]);
                    }
                }
            }
            ssync_setup();
            ht = ht1; cnt = cnt1; ht1 = tslot[it & 1];
        }
        {   // sentinel unit: tells the loader, the MMA thread and (through it) the epilogue to stop
            BmDesc* d = &desc[unit % kBmDescRing];
            mbar_wait(&w_free[0], (unit & 1) ^ 1);
            mbar_wait(&w_free[1], (unit & 1) ^ 1);
            if (st == 0) {
                d->flags = 1; d->j0 = d->j1 = 0; d->nrows = 0;
                __threadfence_block();
                mbar_arrive(&w_ready[0]);
                mbar_arrive(&w_ready[1]);
            }
        }
    }

#ifdef QR_PROF
    if (tid == 0) atomicAdd(&p.sl.ctrl[27], (int)((clock64() - t_start) >> 10));
    if (lane == 0)
        for (int c = 0; c < 11; ++c)
            if (bpw[c]) atomicAdd(&p.sl.ctrl[16 + c], (int)(bpw[c] >> 10));
#endif
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
}

bool backward_mma_supported(int32_t K, int32_t D) { return tc_channels_supported(D) && K >= 1 && K <= QR_MAX_K; }

// workspace = the common layout of qr_sel.cuh (the forward's workspace has the same one)
size_t backward_mma_workspace_bytes(const Cam& cam, int K) { return ws_layout(cam, K).total; }
// points p at the lists and the clear cache inside ws
int backward_mma_workspace_view(BackwardParams& p, void* ws, size_t ws_bytes, int32_t** seen, int* seen_cells)
{
    const WsLayout wl = ws_layout(p.cam, p.K);
    if (ws_bytes < wl.total) return fail(QR_ERR_WORKSPACE_TOO_SMALL, "workspace %zu < %zu bytes", ws_bytes, wl.total);
    if (!aligned16(ws)) return fail(QR_ERR_MISALIGNED, "workspace alignment");
    p.sl = sel_view(wl.sel, ws);
    p.prep_nflag = reinterpret_cast<const int32_t*>(ws);
    *seen = reinterpret_cast<int32_t*>(static_cast<char*>(ws) + wl.seen);
    *seen_cells = kSeenCells;
    return QR_OK;
}

// ------------------------------------------------------------------------------------------------------------------
// backward_prep_kernel: one CTA per half tile, thread = pixel (the pixel order of the MMA's K dimension).  Numbers
// the distinct selected Gaussians of the half tile (shared-memory hash set) and rewrites the selection as entries
// {weight, union row << 8 | pixel} ordered by pixel.  This is the latency-bound, irregular part of qr_backward; run
// here with a dozen CTAs per SM it costs a few microseconds, inside the persistent kernel it was the bottleneck
// (profiles/README.md, r1_c).
// ------------------------------------------------------------------------------------------------------------------
constexpr int kBmPrepThreads = 256;
constexpr int kBmPrepSmem = kBmHash * 4 + kBmHash * 2 + kBmEntCap * 4 + kBmEntCap * 4 + kBmEntCap + 2 * (kBmPx + 4) * 4;

__global__ void __launch_bounds__(kBmPrepThreads) backward_prep_kernel(const BackwardParams p, int32_t* __restrict__ nflag)
{
    extern __shared__ __align__(16) unsigned char psm[];
    int32_t* hkey = reinterpret_cast<int32_t*>(psm);
    int32_t* sid = hkey + kBmHash;
    float* sw = reinterpret_cast<float*>(sid + kBmEntCap);
    int32_t* E = reinterpret_cast<int32_t*>(sw + kBmEntCap);        // [kBmPx + 4] exclusive scan of n_sel
    int32_t* nss = E + kBmPx + 4;                                   // [kBmPx + 4] clamped n_sel
    uint16_t* hslot = reinterpret_cast<uint16_t*>(nss + kBmPx + 4);
    uint8_t* spx = reinterpret_cast<uint8_t*>(hslot + kBmHash);
    __shared__ int32_t warp_sums[kBmPx / 32];
    __shared__ int32_t ucount;
    // threads 0..127 own a pixel each for the scan; all kBmPrepThreads share the record-parallel phases
    const int ht = blockIdx.x, pl = threadIdx.x, lane = pl & 31, warp = pl >> 5;
    const int K = p.K;
    int32_t* hdr = p.sl.hdr + (size_t)ht * kHdrWords;
    if (ht == 0 && pl == 0) {
        p.sl.stamp[0] = kSelMagic; p.sl.stamp[1] = p.cam.width; p.sl.stamp[2] = p.cam.height; p.sl.stamp[3] = K;
        const unsigned long long a = (unsigned long long)p.sel_idx;
        p.sl.stamp[4] = (int32_t)(a & 0xffffffffull); p.sl.stamp[5] = (int32_t)(a >> 32);
    }
    const int tile = ht >> 1;
    const int x0 = (tile % p.cam.tiles_x) * kTile, y0 = (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8;
    // pixel pl of the half tile: stage j = pl >> 3 covers row j >> 1, x = 8 (j & 1) .. + 7
    auto pix_of = [&](int q, int64_t& pix) -> bool {
        const int j = q >> 3, x = x0 + (j & 1) * kBmStagePx + (q & 7), y = y0 + (j >> 1);
        pix = (int64_t)y * p.cam.width + x;
        return x < p.cam.width && y < p.cam.height;
    };
    int64_t pix;
    const bool valid = pl < kBmPx && pix_of(pl, pix);
    const int ns = valid ? max(0, min(K, __ldg(p.n_sel + pix))) : 0;
    int inc = ns;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
    if (lane == 31 && warp < kBmPx / 32) warp_sums[warp] = inc;
    if (pl == 0) ucount = 0;
    __syncthreads();
    int e0 = inc - ns, R = 0, R0 = 0;
#pragma unroll
    for (int w = 0; w < kBmPx / 32; ++w) {
        const int s = warp_sums[w];
        if (w < warp) e0 += s;
        if (w < 2) R0 += s;
        R += s;
    }
    if (R > kBmEntCap || R == 0) {
        if (pl < kHdrWords) hdr[pl] = (pl == 5 && R > kBmEntCap) ? 1 : 0;      // empty lists; [5]: left to the FFMA kernel
        if (pl == 0 && R > kBmEntCap) atomicAdd(nflag, 1);
        return;
    }
    if (pl < kBmPx) { E[pl] = e0; nss[pl] = ns; }
    int hs = 64;
    while (hs < 2 * R) hs <<= 1;
    hs = min(hs, kBmHash);                      // R <= kBmEntCap < kBmHash: the probe loops below always terminate
    const int hmask = hs - 1;
    for (int k = pl; k < hs; k += kBmPrepThreads) hkey[k] = -1;
    __syncthreads();
    // stage the records, thread = record: every load of the half tile is in flight at once, and consecutive
    // threads read consecutive slots of a pixel's list
    for (int s = 0; s < ns; ++s) spx[e0 + s] = (uint8_t)pl;
    __syncthreads();
    for (int k0 = pl; k0 < R; k0 += 8 * kBmPrepThreads) {
        int32_t id[8];
        float w[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int k = k0 + u * kBmPrepThreads;
            id[u] = -1; w[u] = 0.0f;
            if (k < R) {
                const int q = spx[k];
                int64_t pq;
                pix_of(q, pq);
                const int64_t a = pq * K + (k - E[q]);
                id[u] = __ldg(p.sel_idx + a);
                w[u] = __ldg(p.sel_w + a);
            }
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int k = k0 + u * kBmPrepThreads;
            if (k < R) { sid[k] = id[u]; sw[k] = w[u]; }
        }
    }
    __syncthreads();
    int32_t* uid_h = p.sl.uid + (size_t)ht * p.sl.ucap;
#pragma unroll 4
    for (int k = pl; k < R; k += kBmPrepThreads) {       // the thread that creates a cell numbers it
        const int32_t id = sid[k];
        uint32_t h = hash32((uint32_t)id) & hmask;
        while (true) {
            const int32_t old = atomicCAS(&hkey[h], -1, id);
            if (old == -1) {
                const int slot = atomicAdd(&ucount, 1);
                hslot[h] = (uint16_t)slot;
                uid_h[slot] = id;
                break;
            }
            if (old == id) break;
            h = (h + 1) & hmask;
        }
    }
    __syncthreads();
    // the records are ordered by pixel: list q (pixels 32 q .. 32 q + 31) is records [E[32 q], E[32 q + 32])
    uint2* ent_h = p.sl.ent + (size_t)ht * kSelLists * p.sl.qcap;
#pragma unroll 4
    for (int k = pl; k < R; k += kBmPrepThreads) {
        const int32_t id = sid[k];
        uint32_t h = hash32((uint32_t)id) & hmask;
        while (hkey[h] != id) h = (h + 1) & hmask;
        const int q = spx[k], list = q >> 5;
        ent_h[(size_t)list * p.sl.qcap + (k - E[32 * list])] =
            make_uint2(__float_as_uint(sw[k]), sel_pack((int)hslot[h], k - E[q], q));
    }
    if (pl < kHdrWords) {
        int v = 0;
        if (pl < 3) v = E[32 * (pl + 1)] - E[32 * pl];
        else if (pl == 3) v = R - E[96];
        else if (pl == 4) v = ucount;
        hdr[pl] = v;
    }
}

int launch_backward_prep(const BackwardParams& p, int32_t* nflag, cudaStream_t st)
{
    const int num_half = p.cam.tiles_x * p.cam.tiles_y * 2;
    QR_CUDA_OK(cudaFuncSetAttribute(backward_prep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kBmPrepSmem));
    backward_prep_kernel<<<(unsigned)num_half, kBmPrepThreads, kBmPrepSmem, st>>>(p, nflag);
    QR_LAUNCH_OK("backward_prep_kernel");
    return QR_OK;
}

int launch_backward_mma(BackwardParams p, void* ws, size_t ws_bytes, cudaStream_t st, bool from_lists)
{
    const WsLayout wl = ws_layout(p.cam, p.K);
    if (!ws) return fail(QR_ERR_NULL_POINTER, "qr_backward: workspace is NULL");
    if (ws_bytes < wl.total) return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_backward: workspace %zu < %zu bytes", ws_bytes, wl.total);
    if (!aligned16(ws)) return fail(QR_ERR_MISALIGNED, "qr_backward: workspace alignment");
    p.sl = sel_view(wl.sel, ws);
    int32_t* nflag = reinterpret_cast<int32_t*>(ws);
    p.prep_nflag = nflag;
    QR_CUDA_OK(cudaMemsetAsync(nflag, 0, 256, st));      // [0] half tiles left to the FFMA kernel, [1] the contraction's half-tile ticket
    p.ticket = nflag + 1;
    const int sms = sm_count();
    // dL_dmap [H][W][D] fp32 as a 4-D tensor (32 channels, W, D / 32 channel groups, H); box = 32 channels x 8 pixels x
    // all groups x 1 row, 32-byte-atom 128-byte swizzle (what UMMA calls SWIZZLE_128B_BASE32B); pixels outside the image
    // are filled with zeros
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return fail(QR_ERR_CUDA, "qr_backward: cuTensorMapEncodeTiled is not available from the driver");
    CUtensorMap tmap;
    // (D below 128-channel tiles: the box still spans whole tiles, what lies beyond D -- whole 32-channel groups, or the channels
    // behind D < 32 -- is out of bounds for the tensor and arrives as zeros)
    const int Dp = bm_pad(p.D);
    const cuuint64_t dims[4] = { (cuuint64_t)min(32, p.D), (cuuint64_t)p.cam.width, (cuuint64_t)((p.D + 31) / 32), (cuuint64_t)p.cam.height };
    const cuuint64_t strides[3] = { (cuuint64_t)p.D * 4, 128, (cuuint64_t)p.D * 4 * (cuuint64_t)p.cam.width };
    const cuuint32_t box[4] = { 32, kBmStagePx, (cuuint32_t)(Dp / 32), 1 };
    const cuuint32_t estr[4] = { 1, 1, 1, 1 };
    const CUresult cr = enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, const_cast<float*>(p.dL_dmap), dims, strides, box, estr,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) return fail(QR_ERR_CUDA, "qr_backward: cuTensorMapEncodeTiled failed (%d)", (int)cr);
    const int num_half = p.cam.tiles_x * p.cam.tiles_y * 2;
    const unsigned grid = (unsigned)min(sms, num_half);
    const int fixed = bm_smem(Dp, 0).total;
    const int stages = max(2, min(12, (232448 - fixed - 1280) / (kBmStagePx * Dp * 4)));
    const int smem = bm_smem(Dp, stages).total;
    if (!from_lists)
        if (int rc = launch_backward_prep(p, nflag, st)) return rc;
    QR_CUDA_OK(cudaFuncSetAttribute(backward_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    backward_mma_kernel<<<grid, kBmThreads, smem, st>>>(p, stages, tmap);
    QR_LAUNCH_OK("backward_mma_kernel");
    if (from_lists) return QR_OK;       // the walk's lists have exact capacities: no half tile is left over
    // half tiles with more than kBmEntCap records (rare: a mean of more than 24 selections per pixel)
    p.only_flagged = true;
    return launch_backward_tile(p, st);
}

}  // namespace qr

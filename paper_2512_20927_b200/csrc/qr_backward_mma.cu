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
//   B = W, K-major, no swizzle: built by the setup warps from the selection records.
// Precision: kind::tf32 truncates fp32 operands to 10 explicit mantissa bits (measured on B200), so the raw G tile IS
// G_hi; converter warps write G_lo = G - trunc(G) next to it, W is split exactly into W_hi + W_lo, and three MMAs
// accumulate G_hi W_hi + G_hi W_lo + G_lo W_hi in fp32 (TMEM).  The dropped G_lo W_lo term and the truncation of the
// lo parts are <= 2^-21 relative per product, 40x below the fp32 tolerance of north_star (1e-4 relative).
//
// One persistent CTA per SM, 14 warps, roles by warp (no role ever waits at a block barrier):
//   warps 0..3    epilogue: tcgen05.ld of the accumulator (lane = channel, column = union row), one coalesced
//                 red.global.add.f32 per (union row, 32 channels)
//   warp  4       one thread issues tcgen05.mma
//   warp  5       loader: TMA tensor copies of dL_dmap into a ring of stages, far ahead of use
//   warps 6..9    converters: G_lo = G - trunc(G), elementwise over a stage (same swizzled offset in the lo buffer)
//   warps 10..13  setup, one unit ahead: number the distinct selected Gaussians of the unit with a shared-memory hash
//                 set and scatter the weights into W (hi, lo).  W is double buffered by halves of the K range (pixels
//                 0..63 / 64..127): half h of the next unit is rebuilt as soon as the MMAs that read it have retired.
// A unit is (half tile, range of 8-pixel stages, pass): the stage range is cut so that the unit's records fit the
// hash set, and a union larger than 64 rows is processed in passes of 64 rows that re-stream the same pixels.
#include <cuda.h>

#include "qr_async.cuh"
#include "qr_backward.cuh"

namespace qr {

using namespace aq;

constexpr int kBmEpiWarps = 4;
constexpr int kBmMmaWarp = 4;
constexpr int kBmLoadWarp = 5;
constexpr int kBmFirstConv = 6;
constexpr int kBmConvWarps = 4;
constexpr int kBmFirstSetup = kBmFirstConv + kBmConvWarps;       // 10
constexpr int kBmSetupWarps = 4;
constexpr int kBmSetupThreads = kBmSetupWarps * 32;
constexpr int kBmThreads = (kBmFirstSetup + kBmSetupWarps) * 32;  // 448
constexpr int kBmPx = 128;                 // half tile: 16 x 8 pixels
constexpr int kBmStagePx = 8;              // one tf32 K step
constexpr int kBmStagesPerUnit = kBmPx / kBmStagePx;   // 16
constexpr int kBmRows = 64;                // union rows per pass = MMA N
constexpr int kBmHalfPx = 64;              // pixels per W half buffer
constexpr int kBmWHalfBytes = kBmRows * kBmHalfPx * 4;           // 16 KB (hi or lo of one half)
constexpr int kBmHash = 4096;
constexpr int kBmCap = 2048;               // staged records per unit (each pixel padded to a multiple of 4);
                                           // 8 px x QR_MAX_K always fits
constexpr int kBmDescRing = 4;

struct BmDesc {
    int32_t ht, j0, j1, nrows, flags;      // flags: 1 = no more work
    int32_t uid[kBmRows];                  // union row (MMA column) -> Gaussian id
};

struct BmSmem {
    int W, stages, hkey, hslot, sid, sw, spx, nsel, E, desc, bars, misc, total;
};
__host__ __device__ inline BmSmem bm_smem(int D, int stages)
{
    BmSmem L;
    int o = 0;
    L.W = o;      o += 2 * 2 * kBmWHalfBytes;                    // [half][hi, lo]
    L.stages = o; o += stages * 2 * kBmStagePx * D * 4;          // [stage][hi, lo], 1 KB aligned
    L.hkey = o;   o += kBmHash * 4;
    L.sid = o;    o += 2 * kBmCap * 4;
    L.sw = o;     o += 2 * kBmCap * 4;
    L.hslot = o;  o += kBmHash * 2;
    L.spx = o;    o += 2 * kBmCap;
    L.nsel = o;   o += 3 * kBmPx * 4;
    L.E = o;      o += 3 * (kBmPx + 4) * 4;
    L.desc = o;   o += kBmDescRing * (int)sizeof(BmDesc);
    o = (o + 15) & ~15;
    L.bars = o;   o += (3 * stages + 8) * 8;
    L.misc = o;   o += 16;                                       // TMEM base, done flag
    L.total = (o + 15) & ~15;
    return L;
}

__device__ __forceinline__ uint32_t bm_hash(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352dU; x ^= x >> 15; x *= 0x846ca68bU; x ^= x >> 16;
    return x;
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
__device__ __forceinline__ void bm_commit(uint64_t* bar)    // arrives when every MMA issued so far by this thread is done
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(s32(bar)) : "memory");
}
__device__ __forceinline__ void bm_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void bm_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// shared-memory matrix descriptor (sm_100): start >> 4 | LBO >> 4 << 16 | SBO >> 4 << 32 | version 1 << 46 | layout << 61
__device__ __forceinline__ uint64_t bm_desc(uint32_t addr, uint32_t lbo, uint32_t sbo, uint32_t layout)
{
    return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)((lbo >> 4) & 0x3FFF) << 16) |
           ((uint64_t)((sbo >> 4) & 0x3FFF) << 32) | ((uint64_t)1 << 46) | ((uint64_t)layout << 61);
}
__device__ __forceinline__ void bm_mma(uint32_t d_tmem, uint64_t a, uint64_t b, uint32_t idesc, bool accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(a), "l"(b), "r"(idesc), "r"((uint32_t)accumulate) : "memory");
}
__device__ __forceinline__ float bm_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xFFFFE000u); }
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
__device__ __forceinline__ void bm_red(float* dst, float v)
{
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(dst), "f"(v) : "memory");
}

__global__ void __launch_bounds__(kBmThreads, 1)
backward_mma_kernel(const BackwardParams p, const int stages, const __grid_constant__ CUtensorMap g_tmap)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    const int D = p.D, K = p.K;
    const BmSmem L = bm_smem(D, stages);
    const int nchunks = D >> 7;                      // 128-channel MMA tiles
    const int stage_half = kBmStagePx * D * 4;       // bytes of a stage's hi (or lo) part
    unsigned char* Wsm = smem + L.W;
    unsigned char* stage_base = smem + L.stages;
    BmDesc* desc = reinterpret_cast<BmDesc*>(smem + L.desc);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bars);
    uint64_t* raw_full = bars;                       // [stages] loader (TMA complete_tx) -> converters
    uint64_t* conv_done = raw_full + stages;         // [stages] converters (4 warp arrivals) -> MMA
    uint64_t* stage_empty = conv_done + stages;      // [stages] MMA (tcgen05.commit) -> loader
    uint64_t* w_ready = stage_empty + stages;        // [2] setup -> MMA, loader (half 0 also publishes the descriptor)
    uint64_t* w_free = w_ready + 2;                  // [2] MMA (tcgen05.commit) -> setup
    uint64_t* tmem_full = w_free + 2;                // [2] MMA (tcgen05.commit) -> epilogue
    uint64_t* tmem_empty = tmem_full + 2;            // [2] epilogue (4 warp arrivals) -> MMA
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L.misc);
    volatile uint32_t* done_flag = reinterpret_cast<volatile uint32_t*>(smem + L.misc + 4);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int num_half = p.cam.tiles_x * p.cam.tiles_y * 2;

    if (tid == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(&raw_full[s], 1); mbar_init(&conv_done[s], kBmConvWarps); mbar_init(&stage_empty[s], 1); }
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
    bm_fence_before();
    __syncthreads();
    bm_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp < kBmEpiWarps) {
        // ================================================= epilogue =================================================
        // thread = channel 32 warp + lane of every 128-channel tile (TMEM lane), columns = union rows of the unit
        auto ld32 = [&](uint32_t taddr, uint32_t (&r)[32]) {
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
                         : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                           "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
                           "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
                           "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                         : "r"(taddr));
        };
        for (int unit = 0;; ++unit) {
            const int buf = unit & 1;
            mbar_wait(&tmem_full[buf], (unit >> 1) & 1);
            bm_fence_after();
            const BmDesc* d = &desc[unit % kBmDescRing];
            if (d->flags & 1) break;
            const int nrows = d->nrows;
            const uint32_t t0 = tmem_base + ((uint32_t)(warp * 32) << 16) + (uint32_t)(buf * 256);
            float* dcol = p.dL_dfeat + warp * 32 + lane;
            for (int m = 0; m < nchunks; ++m) {
                uint32_t ra[32], rb[32];
                ld32(t0 + m * kBmRows, ra);
                if (nrows > 32) ld32(t0 + m * kBmRows + 32, rb);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                if (m == nchunks - 1) {                 // every tcgen05.ld of this accumulator has completed
                    bm_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&tmem_empty[buf]);
                }
#pragma unroll
                for (int c = 0; c < 32; ++c)
                    if (c < nrows) bm_red(dcol + (int64_t)d->uid[c] * D + m * 128, __uint_as_float(ra[c]));
                if (nrows > 32) {
#pragma unroll
                    for (int c = 0; c < 32; ++c)
                        if (32 + c < nrows) bm_red(dcol + (int64_t)d->uid[32 + c] * D + m * 128, __uint_as_float(rb[c]));
                }
            }
        }
    } else if (warp == kBmMmaWarp) {
        // ================================================= MMA issuer ===============================================
        if (lane == 0) {
            // M = 128 channels, N = 64 rows, fp32 accumulate, A and B tf32, A MN-major, B K-major
            const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | (1u << 15) | ((uint32_t)(kBmRows >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
            const uint32_t w0 = s32(Wsm), st0 = s32(stage_base);
            int st = 0;
            for (int unit = 0;; ++unit) {
                const int buf = unit & 1;
                mbar_wait(&w_ready[0], unit & 1);
                const BmDesc* d = &desc[unit % kBmDescRing];
                const int j0 = d->j0, j1 = d->j1, flags = d->flags;
                mbar_wait(&tmem_empty[buf], ((unit >> 1) & 1) ^ 1);
                bm_fence_after();
                if (flags & 1) { bm_commit(&tmem_full[buf]); break; }
                bool have_w1 = false;
                for (int j = j0; j < j1; ++j, ++st) {
                    const int h = j >> 3;
                    if (h == 1 && !have_w1) { mbar_wait(&w_ready[1], unit & 1); have_w1 = true; }
                    const int s = st % stages;
                    mbar_wait(&conv_done[s], (st / stages) & 1);
                    bm_fence_after();
                    const uint32_t a_hi = st0 + s * 2 * stage_half, a_lo = a_hi + stage_half;
                    const uint32_t b_hi = w0 + h * 2 * kBmWHalfBytes + (j & 7) * 256, b_lo = b_hi + kBmWHalfBytes;
                    const uint64_t db_hi = bm_desc(b_hi, 128, kBmHalfPx / 4 * 128, 0);
                    const uint64_t db_lo = bm_desc(b_lo, 128, kBmHalfPx / 4 * 128, 0);
                    for (int m = 0; m < nchunks; ++m) {
                        const uint64_t da_hi = bm_desc(a_hi + m * 4096, 1024, 512, 1);
                        const uint64_t da_lo = bm_desc(a_lo + m * 4096, 1024, 512, 1);
                        const uint32_t d_tmem = tmem_base + (uint32_t)(buf * 256 + m * kBmRows);
                        bm_mma(d_tmem, da_hi, db_hi, idesc, j != j0);
                        bm_mma(d_tmem, da_hi, db_lo, idesc, true);
                        bm_mma(d_tmem, da_lo, db_hi, idesc, true);
                    }
                    bm_commit(&stage_empty[s]);
                    if (h == 0 && (j == 7 || j == j1 - 1)) bm_commit(&w_free[0]);     // last read of W half 0
                }
                if (!have_w1) mbar_wait(&w_ready[1], unit & 1);       // keep the phases of every unit in step
                if (j0 >= 8) bm_commit(&w_free[0]);
                bm_commit(&w_free[1]);
                bm_commit(&tmem_full[buf]);
            }
        }
    } else if (warp == kBmLoadWarp) {
        // ================================================= loader ===================================================
        // lane c < D / 32 copies channels [32 c, 32 c + 32) of the stage's 8 pixels: a [8 px][128 B] swizzled block
        int st = 0;
        for (int unit = 0;; ++unit) {
            mbar_wait(&w_ready[0], unit & 1);
            const BmDesc* d = &desc[unit % kBmDescRing];
            const int ht = d->ht, j0 = d->j0, j1 = d->j1, flags = d->flags;
            if (flags & 1) {
                const int s = st % stages;
                mbar_wait(&stage_empty[s], ((st / stages) & 1) ^ 1);
                if (lane == 0) { *done_flag = 1u; mbar_arrive(&raw_full[s]); }     // wakes the converters up to stop
                break;
            }
            const int tile = ht >> 1;
            const int x0 = (tile % p.cam.tiles_x) * kTile, y0 = (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8;
            for (int j = j0; j < j1; ++j, ++st) {
                const int s = st % stages;
                mbar_wait(&stage_empty[s], ((st / stages) & 1) ^ 1);
                if (lane == 0) mbar_arrive_expect_tx(&raw_full[s], (uint32_t)stage_half);
                __syncwarp();
                if (lane < (D >> 5))
                    bm_tma_box(stage_base + (size_t)s * 2 * stage_half + lane * 1024, &g_tmap, lane * 32,
                               x0 + (j & 1) * kBmStagePx, y0 + (j >> 1), &raw_full[s]);
            }
        }
    } else if (warp < kBmFirstSetup) {
        // ================================================= converters ===============================================
        const int ct = tid - kBmFirstConv * 32;              // 0..127
        const int n4 = stage_half >> 4;                      // float4 per stage half
        for (int st = 0;; ++st) {
            const int s = st % stages;
            mbar_wait(&raw_full[s], (st / stages) & 1);
            if (*done_flag) break;
            const float4* hi = reinterpret_cast<const float4*>(stage_base + (size_t)s * 2 * stage_half);
            float4* lo = reinterpret_cast<float4*>(stage_base + (size_t)s * 2 * stage_half + stage_half);
#pragma unroll 4
            for (int i = ct; i < n4; i += kBmConvWarps * 32) {
                const float4 v = hi[i];
                lo[i] = make_float4(__fsub_rn(v.x, bm_hi(v.x)), __fsub_rn(v.y, bm_hi(v.y)), __fsub_rn(v.z, bm_hi(v.z)),
                                    __fsub_rn(v.w, bm_hi(v.w)));
            }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(&conv_done[s]);
        }
    } else {
        // ================================================= setup ====================================================
        // Software pipeline over this CTA's half tiles h_0, h_1, ...: while h_i is hashed and scattered out of shared
        // memory, the selection records of h_(i+1) and the n_sel of h_(i+2) are in flight (cp.async), so no
        // global-load latency sits on the path that feeds the MMAs.
        const int st = tid - kBmFirstSetup * 32;          // 0..127
        int32_t* hkey = reinterpret_cast<int32_t*>(smem + L.hkey);
        uint16_t* hslot = reinterpret_cast<uint16_t*>(smem + L.hslot);
        int32_t* sid_all = reinterpret_cast<int32_t*>(smem + L.sid);
        float* sw_all = reinterpret_cast<float*>(smem + L.sw);
        uint8_t* spx_all = smem + L.spx;
        int32_t* nsel_all = reinterpret_cast<int32_t*>(smem + L.nsel);
        int32_t* E_all = reinterpret_cast<int32_t*>(smem + L.E);
        __shared__ int32_t ucount;
        const bool k4 = (K & 3) == 0;
        auto ssync = [&]() { named_sync<1, kBmSetupThreads>(); };
        auto origin = [&](int ht, int& x0, int& y0) {
            const int tile = ht >> 1;
            x0 = (tile % p.cam.tiles_x) * kTile;
            y0 = (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8;
        };
        auto next_ht = [&](int ht) {                      // next half tile of this CTA that has rows inside the image
            while (true) {
                ht += gridDim.x;
                if (ht >= num_half) return num_half;
                int x0, y0;
                origin(ht, x0, y0);
                if (y0 < p.cam.height) return ht;
            }
        };
        // pixel pl of a half tile: stage j = pl >> 3 covers row j >> 1, x = 8 (j & 1) .. + 7
        auto pix_of = [&](int x0, int y0, int pl, int64_t& pix) -> bool {
            const int j = pl >> 3, x = x0 + (j & 1) * kBmStagePx + (pl & 7), y = y0 + (j >> 1);
            pix = (int64_t)y * p.cam.width + x;
            return x < p.cam.width && y < p.cam.height;
        };
        auto issue_nsel = [&](int ht, int nb) {           // n_sel of the 128 pixels -> nsel_all[nb] (async)
            if (ht >= num_half) return;
            int x0, y0;
            origin(ht, x0, y0);
            for (int pl = st; pl < kBmPx; pl += kBmSetupThreads) {
                int64_t pix;
                if (pix_of(x0, y0, pl, pix)) bm_cp4(&nsel_all[nb * kBmPx + pl], p.n_sel + pix);
                else nsel_all[nb * kBmPx + pl] = 0;
            }
        };
        auto plan = [&](int nb) {                         // clamp n_sel, E = exclusive scan of the padded counts
            if (st < 32) {
                int32_t* ns = nsel_all + nb * kBmPx + st * 4;
                int v[4], sum = 0;
#pragma unroll
                for (int k = 0; k < 4; ++k) { v[k] = max(0, min(K, ns[k])); ns[k] = v[k]; sum += (v[k] + 3) & ~3; }
                int inc = sum;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (st >= o) inc += t; }
                int e = inc - sum;
                int32_t* E = E_all + nb * (kBmPx + 4) + st * 4;
#pragma unroll
                for (int k = 0; k < 4; ++k) { E[k] = e; e += (v[k] + 3) & ~3; }
                if (st == 31) E_all[nb * (kBmPx + 4) + kBmPx] = e;
            }
            ssync();
        };
        auto range_end = [&](int nb, int j0) {            // as many 8-pixel stages as fit the staging buffers
            const int32_t* E = E_all + nb * (kBmPx + 4);
            int j1 = j0 + 1;
            while (j1 < kBmStagesPerUnit && E[(j1 + 1) * kBmStagePx] - E[j0 * kBmStagePx] <= kBmCap) ++j1;
            return j1;
        };
        auto issue_rec = [&](int ht, int nb, int sb, int j0, int j1) {   // records of stages [j0, j1) -> staging sb
            int x0, y0;
            origin(ht, x0, y0);
            const int32_t* E = E_all + nb * (kBmPx + 4);
            const int base = E[j0 * kBmStagePx];
            int32_t* sid = sid_all + sb * kBmCap;
            float* sw = sw_all + sb * kBmCap;
            uint8_t* spx = spx_all + sb * kBmCap;
            for (int pl = j0 * kBmStagePx + st; pl < j1 * kBmStagePx; pl += kBmSetupThreads) {
                const int ns = nsel_all[nb * kBmPx + pl];
                if (ns == 0) continue;
                int64_t pix;
                pix_of(x0, y0, pl, pix);
                const int o = E[pl] - base;
                const int32_t* gi = p.sel_idx + pix * K;
                const float* gw = p.sel_w + pix * K;
                if (k4) {
                    for (int c = 0; c < ns; c += 4) {
                        bm_cp16(sid + o + c, gi + c);
                        bm_cp16(sw + o + c, gw + c);
                        *reinterpret_cast<uint32_t*>(spx + o + c) = (uint32_t)pl * 0x01010101u;
                    }
                } else {
                    for (int c = 0; c < ns; ++c) {
                        bm_cp4(sid + o + c, gi + c);
                        bm_cp4(sw + o + c, gw + c);
                        spx[o + c] = (uint8_t)pl;
                    }
                }
            }
        };
        auto fixup = [&](int nb, int sb, int j0, int j1) {   // padding entries of every pixel: id -1
            const int32_t* E = E_all + nb * (kBmPx + 4);
            const int base = E[j0 * kBmStagePx];
            int32_t* sid = sid_all + sb * kBmCap;
            for (int pl = j0 * kBmStagePx + st; pl < j1 * kBmStagePx; pl += kBmSetupThreads) {
                const int ns = nsel_all[nb * kBmPx + pl];
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
        bm_cp_wait_all();
        ssync();
        if (ht < num_half) {
            plan(0);
            issue_rec(ht, 0, 0, 0, range_end(0, 0));
            issue_nsel(ht1, 1);
        }
        for (int i = 0; ht < num_half; ++i) {
            const int nb = i % 3, sb = i & 1;
            const int32_t* E = E_all + nb * (kBmPx + 4);
            bm_cp_wait_all();
            ssync();                                      // records(h_i, first range) and n_sel(h_(i+1)) have landed
            const int ht2 = ht1 < num_half ? next_ht(ht1) : num_half;
            if (ht1 < num_half) {
                const int nb1 = (i + 1) % 3;
                plan(nb1);
                issue_rec(ht1, nb1, sb ^ 1, 0, range_end(nb1, 0));
                issue_nsel(ht2, (i + 2) % 3);
            }
            int j0 = 0;
            while (j0 < kBmStagesPerUnit) {
                const int j1 = range_end(nb, j0);
                const int base = E[j0 * kBmStagePx];
                const int R = E[j1 * kBmStagePx] - base;
                if (R == 0) { j0 = j1; continue; }                  // nothing selected in these stages: no unit
                if (j0 > 0) {                                      // later range of the same half tile (rare)
                    ssync();
                    issue_rec(ht, nb, sb, j0, j1);
                    bm_cp_wait_all();
                    ssync();
                }
                fixup(nb, sb, j0, j1);
                int hs = 64;
                while (hs < 2 * R) hs <<= 1;
                hs = min(hs, kBmHash);
                const int hmask = hs - 1;
                {
                    int4* hz = reinterpret_cast<int4*>(hkey);
                    for (int k = st; k < hs / 4; k += kBmSetupThreads) hz[k] = make_int4(-1, -1, -1, -1);
                }
                if (st == 0) ucount = 0;
                ssync();
                const int32_t* sid = sid_all + sb * kBmCap;
                const float* sw = sw_all + sb * kBmCap;
                const uint8_t* spx = spx_all + sb * kBmCap;
                // ---- insert the ids; the thread that creates a cell numbers it ----
                for (int k = st; k < R; k += kBmSetupThreads) {
                    const int32_t id = sid[k];
                    if (id < 0) continue;
                    uint32_t h = bm_hash((uint32_t)id) & hmask;
                    while (true) {
                        const int32_t old = atomicCAS(&hkey[h], -1, id);
                        if (old == -1) { hslot[h] = (uint16_t)atomicAdd(&ucount, 1); break; }
                        if (old == id) break;
                        h = (h + 1) & hmask;
                    }
                }
                ssync();
                const int U = ucount;
                const int npass = (U + kBmRows - 1) / kBmRows;
                // records of W half h: pixels [max(8 j0, 64 h), min(8 j1, 64 h + 64))
                int kb[3];
                kb[0] = 0;
                kb[1] = E[min(max(kBmHalfPx, j0 * kBmStagePx), j1 * kBmStagePx)] - base;
                kb[2] = R;
                for (int pass = 0; pass < npass; ++pass, ++unit) {
                    BmDesc* d = &desc[unit % kBmDescRing];
                    for (int h = 0; h < 2; ++h) {
                        mbar_wait(&w_free[h], (unit & 1) ^ 1);      // the MMAs of the previous unit have read this half
                        float4* wz = reinterpret_cast<float4*>(Wsm + h * 2 * kBmWHalfBytes);
                        for (int k = st; k < 2 * kBmWHalfBytes / 16; k += kBmSetupThreads) wz[k] = make_float4(0.f, 0.f, 0.f, 0.f);
                        ssync();
                        unsigned char* whi = Wsm + h * 2 * kBmWHalfBytes;
                        for (int k = kb[h] + st; k < kb[h + 1]; k += kBmSetupThreads) {
                            const int32_t id = sid[k];
                            if (id < 0) continue;
                            uint32_t hh = bm_hash((uint32_t)id) & hmask;
                            while (hkey[hh] != id) hh = (hh + 1) & hmask;
                            const int c = (int)hslot[hh] - pass * kBmRows;
                            if (c >= 0 && c < kBmRows) {
                                const uint32_t off = bm_w_off(c, (int)spx[k] & (kBmHalfPx - 1));
                                const float w = sw[k], hi = bm_hi(w);
                                *reinterpret_cast<float*>(whi + off) = hi;
                                *reinterpret_cast<float*>(whi + kBmWHalfBytes + off) = __fsub_rn(w, hi);
                                d->uid[c] = id;
                            }
                        }
                        if (h == 0 && st == 0) {
                            d->ht = ht; d->j0 = j0; d->j1 = j1; d->flags = 0;
                            d->nrows = min(kBmRows, U - pass * kBmRows);
                        }
                        fence_async_smem();                        // W is read by the tensor core (async proxy)
                        __threadfence_block();
                        ssync();
                        if (st == 0) mbar_arrive(&w_ready[h]);
                    }
                }
                j0 = j1;
            }
            ht = ht1; ht1 = ht2;
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

    bm_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
}

bool backward_mma_supported(int32_t K, int32_t D) { return D % 128 == 0 && D >= 128 && D <= 512 && K >= 1 && K <= QR_MAX_K; }

typedef CUresult (*BmEncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                    const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static BmEncodeTiledFn bm_encode_tiled_fn()
{
    static BmEncodeTiledFn fn = nullptr;
    if (!fn) {
        void* sym = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<BmEncodeTiledFn>(sym);
    }
    return fn;
}

int launch_backward_mma(const BackwardParams& p, cudaStream_t st)
{
    static int sms = 0;
    if (sms == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
            sms = 148;
    }
    // dL_dmap [H][W][D] fp32 as a 3-D tensor (D, W, H); box = 32 channels x 8 pixels x 1 row, 32-byte-atom 128-byte
    // swizzle (what UMMA calls SWIZZLE_128B_BASE32B); pixels outside the image are filled with zeros
    BmEncodeTiledFn enc = bm_encode_tiled_fn();
    if (!enc) return fail(QR_ERR_CUDA, "qr_backward: cuTensorMapEncodeTiled is not available from the driver");
    CUtensorMap tmap;
    const cuuint64_t dims[3] = { (cuuint64_t)p.D, (cuuint64_t)p.cam.width, (cuuint64_t)p.cam.height };
    const cuuint64_t strides[2] = { (cuuint64_t)p.D * 4, (cuuint64_t)p.D * 4 * (cuuint64_t)p.cam.width };
    const cuuint32_t box[3] = { 32, kBmStagePx, 1 };
    const cuuint32_t estr[3] = { 1, 1, 1 };
    const CUresult cr = enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(p.dL_dmap), dims, strides, box, estr,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) return fail(QR_ERR_CUDA, "qr_backward: cuTensorMapEncodeTiled failed (%d)", (int)cr);
    const int num_half = p.cam.tiles_x * p.cam.tiles_y * 2;
    const unsigned grid = (unsigned)min(sms, num_half);
    const int fixed = bm_smem(p.D, 0).total;
    const int stages = max(2, min(8, (232448 - fixed - 1280) / (2 * kBmStagePx * p.D * 4)));
    const int smem = bm_smem(p.D, stages).total;
    QR_CUDA_OK(cudaFuncSetAttribute(backward_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    backward_mma_kernel<<<grid, kBmThreads, smem, st>>>(p, stages, tmap);
    QR_LAUNCH_OK("backward_mma_kernel");
    return QR_OK;
}

}  // namespace qr

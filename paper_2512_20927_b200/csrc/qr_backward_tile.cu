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
constexpr int kBtThreads = 384;           // warps 0..7 consumers, 8..10 setup, 11 loader
constexpr int kBtConsumerRegs = 216;
constexpr int kBtProducerRegs = 72;
constexpr int kBtPx = 128;                // half tile: 16 x 8 pixels
constexpr int kBtStagePx = 8;
constexpr int kBtStagesPerUnit = kBtPx / kBtStagePx;   // 16
constexpr int kBtRows = 64;               // union rows per pass
constexpr int kBtWStride = 72;            // words per pixel of W: 4 pixels x 8 rows fall into 32 distinct banks
constexpr int kBtHash = 4096;
constexpr int kBtMaxRec = 2800;           // records per unit (hash load <= 0.7); 8 px x QR_MAX_K = 2048 always fits

struct BtDesc {
    int32_t ht, j0, j1, nrows, flags;     // flags: 1 = no more work
    int32_t uid[kBtRows];                 // column (w * 8 + r) -> Gaussian id
};

struct BtSmem {
    int ring, W, hkey, hslot, nsel, ssum, desc, bars, total;
};
__host__ __device__ inline BtSmem bt_smem(int D, int stages)
{
    BtSmem L;
    int o = 0;
    L.ring = o;  o += stages * kBtStagePx * D * 4;
    L.W = o;     o += 2 * kBtPx * kBtWStride * 4;
    L.hkey = o;  o += kBtHash * 4;
    L.hslot = o; o += kBtHash * 2;
    L.nsel = o;  o += kBtPx * 4;
    L.ssum = o;  o += kBtStagesPerUnit * 4;
    L.desc = o;  o += 2 * (int)sizeof(BtDesc);
    o = (o + 15) & ~15;
    L.bars = o;  o += (2 * stages + 4) * 8;
    L.total = (o + 15) & ~15;
    return L;
}

__device__ __forceinline__ uint32_t bt_hash(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352dU; x ^= x >> 15; x *= 0x846ca68bU; x ^= x >> 16;
    return x;
}

__device__ __forceinline__ void bt_red4(float* dst, const float2& a, const float2& b)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y) : "memory");
}

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
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kBtProducerRegs));
        if (warp == kBtConsumers + kBtSetupWarps) {
            // ================================================ loader ================================================
            if (lane == 0) {
                int it = 0;
                for (int unit = 0;; ++unit) {
                    const int b = unit & 1;
                    mbar_wait(&unit_full[b], (unit >> 1) & 1);
                    const int ht = desc[b].ht, j0 = desc[b].j0, j1 = desc[b].j1, flags = desc[b].flags;
                    mbar_arrive(&unit_empty[b]);
                    if (flags & 1) break;
                    const int tile = ht >> 1;
                    const int x0 = (tile % p.cam.tiles_x) * kTile, y0 = (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8;
                    for (int j = j0; j < j1; ++j, ++it) {
                        const int s = it % stages;
                        mbar_wait(&empty[s], ((it / stages) & 1) ^ 1);
                        const int x = x0 + (j & 1) * kBtStagePx, y = y0 + (j >> 1);
                        const int npx = y < p.cam.height ? max(0, min(kBtStagePx, p.cam.width - x)) : 0;
                        if (npx > 0) {
                            const uint32_t bytes = (uint32_t)npx * (uint32_t)D * 4u;
                            mbar_arrive_expect_tx(&full[s], bytes);
                            bulk_g2s(ring + (size_t)s * stage_floats, p.dL_dmap + ((int64_t)y * p.cam.width + x) * D, bytes, &full[s]);
                        } else {
                            mbar_arrive(&full[s]);
                        }
                    }
                }
            }
        } else {
            // ================================================ setup =================================================
            const int st = tid - kBtConsumers * 32;      // 0..95
            int32_t* hkey = reinterpret_cast<int32_t*>(smem + L.hkey);
            uint16_t* hslot = reinterpret_cast<uint16_t*>(smem + L.hslot);
            int32_t* nsel_s = reinterpret_cast<int32_t*>(smem + L.nsel);
            int32_t* ssum = reinterpret_cast<int32_t*>(smem + L.ssum);
            __shared__ int32_t ucount;
            auto ssync = [&]() { named_sync<1, kBtSetupThreads>(); };
            int unit = 0;
            for (int ht = blockIdx.x; ht < num_half; ht += gridDim.x) {
                const int tile = ht >> 1;
                const int x0 = (tile % p.cam.tiles_x) * kTile, y0 = (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8;
                if (y0 >= p.cam.height) continue;
                // pixel pl of the half tile: stage j = pl >> 3 covers row j >> 1, x = 8 (j & 1) .. + 7
                auto pix_of = [&](int pl, int64_t& pix) -> bool {
                    const int j = pl >> 3, x = x0 + (j & 1) * kBtStagePx + (pl & 7), y = y0 + (j >> 1);
                    pix = (int64_t)y * p.cam.width + x;
                    return x < p.cam.width && y < p.cam.height;
                };
                for (int pl = st; pl < kBtPx; pl += kBtSetupThreads) {
                    int64_t pix;
                    nsel_s[pl] = pix_of(pl, pix) ? max(0, min(K, __ldg(p.n_sel + pix))) : 0;
                }
                ssync();
                if (st < kBtStagesPerUnit) {
                    int t = 0;
#pragma unroll
                    for (int q = 0; q < kBtStagePx; ++q) t += nsel_s[st * kBtStagePx + q];
                    ssum[st] = t;
                }
                ssync();
                int j0 = 0;
                while (j0 < kBtStagesPerUnit) {
                    // ---- stage range of this unit: as many stages as fit the hash set ----
                    int tot = 0, j1 = j0;
                    while (j1 < kBtStagesPerUnit) {
                        const int s = ssum[j1];
                        if (j1 > j0 && tot + s > kBtMaxRec) break;
                        tot += s; ++j1;
                    }
                    if (tot == 0) { j0 = j1; continue; }             // nothing selected: no unit
                    int hs = 64;
                    while (hs < 2 * tot) hs <<= 1;
                    hs = min(hs, kBtHash);
                    const int hmask = hs - 1;
                    for (int i = st; i < hs; i += kBtSetupThreads) hkey[i] = -1;
                    if (st == 0) ucount = 0;
                    ssync();
                    // ---- insert the ids ----
                    for (int pl = j0 * kBtStagePx + st; pl < j1 * kBtStagePx; pl += kBtSetupThreads) {
                        const int ns = nsel_s[pl];
                        if (ns == 0) continue;
                        int64_t pix;
                        pix_of(pl, pix);
                        const int32_t* ids = p.sel_idx + pix * K;
                        for (int s = 0; s < ns; ++s) {
                            const int32_t id = __ldg(ids + s);
                            uint32_t h = bt_hash((uint32_t)id) & hmask;
                            while (true) {
                                const int32_t old = atomicCAS(&hkey[h], -1, id);
                                if (old == -1 || old == id) break;
                                h = (h + 1) & hmask;
                            }
                        }
                    }
                    ssync();
                    // ---- number the occupied cells ----
                    for (int i = st; i < hs; i += kBtSetupThreads)
                        if (hkey[i] >= 0) hslot[i] = (uint16_t)atomicAdd(&ucount, 1);
                    ssync();
                    const int U = ucount;
                    const int npass = (U + kBtRows - 1) / kBtRows;
                    for (int pass = 0; pass < npass; ++pass, ++unit) {
                        const int b = unit & 1;
                        mbar_wait(&unit_empty[b], ((unit >> 1) & 1) ^ 1);
                        float* Wb = Wbuf + b * kBtPx * kBtWStride;
                        {
                            float4* wz = reinterpret_cast<float4*>(Wb + j0 * kBtStagePx * kBtWStride);
                            const int n4 = (j1 - j0) * kBtStagePx * kBtWStride / 4;
                            for (int i = st; i < n4; i += kBtSetupThreads) wz[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                        }
                        ssync();
                        for (int pl = j0 * kBtStagePx + st; pl < j1 * kBtStagePx; pl += kBtSetupThreads) {
                            const int ns = nsel_s[pl];
                            if (ns == 0) continue;
                            int64_t pix;
                            pix_of(pl, pix);
                            const int32_t* ids = p.sel_idx + pix * K;
                            const float* ws = p.sel_w + pix * K;
                            for (int s = 0; s < ns; ++s) {
                                const int32_t id = __ldg(ids + s);
                                const float w = __ldg(ws + s);
                                uint32_t h = bt_hash((uint32_t)id) & hmask;
                                while (hkey[h] != id) h = (h + 1) & hmask;
                                const int c = (int)hslot[h] - pass * kBtRows;
                                if (c >= 0 && c < kBtRows) {
                                    const int col = (c & 7) * 8 + (c >> 3);      // consumer warp c % 8, its row c / 8
                                    Wb[pl * kBtWStride + col] = w;
                                    desc[b].uid[col] = id;
                                }
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
                ssync();                                   // nsel_s / ssum are rewritten by the next half tile
            }
            {
                const int b = unit & 1;
                mbar_wait(&unit_empty[b], ((unit >> 1) & 1) ^ 1);
                if (st == 0) { desc[b].flags = 1; desc[b].j0 = desc[b].j1 = 0; __threadfence_block(); mbar_arrive(&unit_full[b]); }
            }
        }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kBtConsumerRegs));
        // ================================================== consumers ===============================================
        float2 acc[8][NV][2];
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int j = 0; j < NV; ++j) acc[r][j][0] = acc[r][j][1] = make_float2(0.f, 0.f);
        int it = 0;
        for (int unit = 0;; ++unit) {
            const int b = unit & 1;
            mbar_wait(&unit_full[b], (unit >> 1) & 1);
            const BtDesc* d = &desc[b];
            if (d->flags & 1) break;
            const int j0 = d->j0, j1 = d->j1, nrows = d->nrows;
            const float* Wb = Wbuf + b * kBtPx * kBtWStride + warp * 8 + (lane & 7) + (lane >> 3) * kBtWStride;
            for (int j = j0; j < j1; ++j, ++it) {
                const int s = it % stages;
                mbar_wait(&full[s], (it / stages) & 1);
                const float* gs = ring + (size_t)s * stage_floats + lane * 4;
#pragma unroll
                for (int hq = 0; hq < 2; ++hq) {
                    // lane = (pixel hq*4 + (lane >> 3) of the stage, row lane & 7 of this warp)
                    const float wl = Wb[(j * kBtStagePx + hq * 4) * kBtWStride];
                    const uint32_t m32 = __ballot_sync(0xffffffffu, wl != 0.0f);
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
#pragma unroll
                        for (int r = 0; r < 8; ++r) {
                            if (m & (1u << r)) {
                                const float w = __shfl_sync(0xffffffffu, wl, q * 8 + r);
                                const float2 ww = make_float2(w, w);
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
    static int sms = 0;
    if (sms == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
            sms = 148;
    }
    const int num_half = p.cam.tiles_x * p.cam.tiles_y * 2;
    const unsigned grid = (unsigned)min(sms, num_half);
    const int stages = p.D >= 512 ? 5 : (p.D >= 256 ? 8 : 12);
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

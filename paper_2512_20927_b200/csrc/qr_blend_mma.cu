// qr_blend_mma.cu -- the O(KC) blend of qr_forward (Algorithm 1 lines 9 and 20) as a dense
// contraction on the 5th-generation tensor cores.
//
// Per 16x8-pixel half tile the blend is  out[128 px, D] = W[128 px, U] . F[U, D]  with U the union of the Gaussians
// selected by any of the 128 pixels (mean 47, 23 % dense at config 3) and W the sparse, already normalised weights
// w^Q / (1 - T^Q) that walk2_kernel left as entry lists (qr_sel.cuh).  ncu showed the FFMA formulation of this product
// to be issue bound at 3x the time of its HBM traffic (profiles/README.md, r1_a), which is the evidence north_star asks
// for before putting it on tensor cores.
//
// Precision: kind::tf32 truncates its fp32 operands to 10 explicit mantissa bits (measured on B200), so both operands
// are split exactly, x = hi + lo with hi = x & 0xFFFFE000 and lo = x - hi, and three MMAs accumulate
// W_hi F_hi + W_lo F_hi + W_hi F_lo in fp32 (TMEM).  The dropped W_lo F_lo term and the truncation of the lo parts
// are <= 2^-21 relative per product, 40x below the fp32 tolerance of north_star (1e-4 relative).
//
// One persistent CTA per SM, 16 warps (512 threads, <= 64 registers, ~155 KB of shared memory: the kernel is meant to
// share its SM with CTAs of walk2_kernel, which it follows by programmatic dependent launch), roles by warp, no role
// ever waits at a block barrier:
//   warps 0..3    epilogue: tcgen05.ld of the accumulator (thread = pixel), st.shared into a 128-byte-swizzled staging
//                 tile, one TMA tensor store per (32 pixels x 32 channels): the map leaves the SM as whole 128-byte lines
//   warp  4       MMA issue: warp-uniform loop, one elected lane issues tcgen05.mma (M = 128 pixels, N = 128 channels,
//                 K = 8 union rows per instruction; A = W from TENSOR MEMORY, B = features from shared memory)
//   warps 5..7    loaders (stage st belongs to warp 5 + st % 3: issuing the copies was the pipeline's bottleneck with one
//                 warp): one bulk async copy (TMA) per 512-byte feature row quarter into a 12-deep raw ring
//   warps 8..11   converters: ld.shared of a raw row -> hi/lo split -> st.shared in the MN-major
//                 SWIZZLE_128B_BASE32B layout tf32 needs for a row-major (channel-contiguous) B operand
//   warps 12..15  builders: claim the next half tile (global ticket, same order as the walk), wait for its ready flag,
//                 publish its descriptor to the other roles; scatter the entry lists into a [128 px][64 col] scratch tile
//                 in shared memory (thread = entry), then, thread = pixel = TMEM lane, read the pixel's row back, split
//                 it and tcgen05.st it into one of two W buffers in tensor memory.  W never sits in shared memory while
//                 the MMAs run, and the build of half tile i + 1 overlaps all of half tile i.
// Tensor memory: columns [0, 256) two 128-column accumulators (the MMAs of unit i+1 overlap the epilogue of unit i),
// [256, 512) two W buffers of 64 hi + 64 lo columns.  Work unit = (half tile, 128 channels).  A half tile whose union
// exceeds 64 columns is processed in rounds of 64 columns (two rounds keep both W instances resident).
#include <cuda.h>
#include <stdlib.h>

#include "qr_blend.cuh"
#include "qr_umma.cuh"

namespace qr {

using namespace aq;

constexpr int kEpiWarps = 4;
constexpr int kMmaWarp = 4;
constexpr int kLoadWarp = 5;                              // warps 5, 6, 7: stage st is loaded by warp 5 + st % 3
constexpr int kLoadWarps = 3;
constexpr int kSchedWarp = 8;
constexpr int kFirstConv = 9;
#ifndef KCONV
#define KCONV 3
#endif
constexpr int kConvWarps = KCONV;                         // stage st is converted by warp 9 + st % kConvWarps
constexpr int kFirstBuild = kFirstConv + kConvWarps;
constexpr int kBuildWarps = 4;
constexpr int kMmaThreads = (kFirstBuild + kBuildWarps) * 32;   // 512
constexpr int kBuildThreads = kBuildWarps * 32;
constexpr int kDescReaders = kEpiWarps + 1 + kLoadWarps + kConvWarps + kBuildWarps;   // warps that read a descriptor
constexpr int kWCols = 64;                                // union columns per round
constexpr int kUnitN = 128;                               // channels per work unit
constexpr int kStageRows = 8;                             // union rows per stage = one tf32 K step
#ifndef KSTAGES
#define KSTAGES 6
#endif
constexpr int kStages = KSTAGES;
#ifndef KRAW
#define KRAW 12
#endif
constexpr int kRawStages = KRAW;
constexpr int kRawRow = kUnitN * 4;                       // 512 B: one feature row quarter
constexpr int kRawBytes = kStageRows * kRawRow;           // 4 KB per raw stage
constexpr int kWsRow = kWCols + 4;                        // scratch row stride in floats: 272 B, conflict-free 16-byte row reads
constexpr int kWsBytes = 128 * kWsRow * 4;                // 34 KB scratch tile
constexpr int kStageHalf = kStageRows * kUnitN * 4;       // 4 KB (hi or lo)
constexpr int kTmemW = 256;                               // first W column in tensor memory
constexpr int kStageBytes = 2 * kStageHalf;
#ifndef KOUTBUFS
#define KOUTBUFS 3
#endif
#ifndef KEBUF
#define KEBUF 512
#endif
constexpr int kOutBufs = KOUTBUFS;                               // staging tiles per epilogue warp
constexpr int kOutTile = 32 * 128;                        // 32 pixels x 32 channels fp32
constexpr int kDescRing = 4;
constexpr int kUidS = 128;                                // union ids per half tile the builders hand to the loader through shared memory
constexpr int kEbuf = KEBUF;                                // entries of each list staged in shared memory (cp.async)

struct MmaDesc { int32_t ht, U, n0, n1, n2, n3, end, pad; };

struct MmaSmem {
    static constexpr int w = 0;                                           // scratch tile [128 px][kWsRow]
    static constexpr int stages = kWsBytes;
    static constexpr int raw = stages + kStages * kStageBytes;
    static constexpr int out = raw + kRawStages * kRawBytes;              // [4 warps][kOutBufs] staging tiles, 1 KB aligned
    static constexpr int ebuf = out + kEpiWarps * kOutBufs * kOutTile;     // uint2[4 lists][kEbuf] staged entries
    static constexpr int desc = ebuf + kSelLists * kEbuf * 8;
    static constexpr int uid = desc + kDescRing * (int)sizeof(MmaDesc);    // int32[kDescRing][kUidS]: first ids of each union
    static constexpr int bars = uid + kDescRing * kUidS * 4;
    static constexpr int n_bars = 2 * kStages + 2 * kRawStages + 4 + 4 + 2 * kDescRing;
    static constexpr int tmem = bars + n_bars * 8;
    static constexpr int total = tmem + 16;
};

__device__ __forceinline__ int32_t ld_acquire(const int32_t* p)
{
    int32_t v;
    asm volatile("ld.acquire.gpu.global.b32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// four rows of the [N, D] feature table, any four, 128 channels each, in one TMA instruction: they land as [4][512 B]
__device__ __forceinline__ void tma_gather4(void* dst, const CUtensorMap* map, int c0, int r0, int r1, int r2, int r3, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cta.global.tile::gather4.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
                 ::"r"(s32(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(s32(bar)), "r"(c0), "r"(r0), "r"(r1), "r"(r2), "r"(r3) : "memory");
}
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* map, const void* src, int c0, int x, int y)
{
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];"
                 ::"l"(reinterpret_cast<uint64_t>(map)), "r"(s32(src)), "r"(c0), "r"(x), "r"(y) : "memory");
}

// rounds / K steps of a half tile: every role derives them from the union size
__device__ __forceinline__ int rounds_of(int U) { return U <= kWCols ? 1 : (U + kWCols - 1) / kWCols; }
__device__ __forceinline__ int cols_of(int U, int r) { return max(0, min(kWCols, U - r * kWCols)); }
__device__ __forceinline__ int ksteps_of(int ncols) { return max(1, (ncols + kStageRows - 1) / kStageRows); }

#ifndef KMINB
#define KMINB 2
#endif
__global__ void __launch_bounds__(kMmaThreads, KMINB)   // "2" only caps the registers at 64; shared memory allows one CTA
blend_mma_kernel(const BlendParams p, const __grid_constant__ CUtensorMap out_tmap, const __grid_constant__ CUtensorMap feat_tmap)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char* stage_base = smem + MmaSmem::stages;
    MmaDesc* desc = reinterpret_cast<MmaDesc*>(smem + MmaSmem::desc);
    int32_t* uid_s = reinterpret_cast<int32_t*>(smem + MmaSmem::uid);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + MmaSmem::bars);
    uint64_t* full = bars;                       // [kStages] converter warp of the stage -> MMA
    uint64_t* empty = bars + kStages;            // [kStages] MMA -> converters (tcgen05.commit)
    uint64_t* raw_full = bars + 2 * kStages;     // [kRawStages] loader (TMA complete_tx) -> converters
    uint64_t* raw_empty = raw_full + kRawStages; // [kRawStages] converter warp of the stage -> loader
    uint64_t* w_ready = raw_empty + kRawStages;  // [2] builders -> MMA: W instance i lives in tensor-memory buffer i & 1
    uint64_t* w_free = w_ready + 2;              // [2] MMA -> builders (tcgen05.commit)
    uint64_t* tmem_full = w_free + 2;            // [2] MMA -> epilogue (tcgen05.commit)
    uint64_t* tmem_empty = tmem_full + 2;        // [2] epilogue -> MMA (4 warp arrivals)
    uint64_t* d_ready = tmem_empty + 2;          // [kDescRing] scheduler -> everybody: descriptor h is published
    uint64_t* d_free = d_ready + kDescRing;      // [kDescRing] every consumer warp, once it has copied descriptor h -> scheduler
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + MmaSmem::tmem);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int D = (p.D + kUnitN - 1) / kUnitN * kUnitN;      // whole 128-channel units; TMA pads the loads and clips the stores
    // fp16 features (R14: widened exactly): a raw row quarter is 256 bytes, the widened value IS the tf32 operand (10 explicit mantissa
    // bits: nothing to split off), so the F_lo buffer is never written and the third MMA is skipped
    const bool f16 = p.feat_f16 != 0;
    const int raw_row = f16 ? kRawRow / 2 : kRawRow;
    const int nunits = D / kUnitN;
    const int num_half = p.num_tiles * 2;

    if (tid == 0) {
        stamp_time(p.sl.ctrl, 2, true);
        for (int s = 0; s < kStages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
        for (int s = 0; s < kRawStages; ++s) { mbar_init(&raw_full[s], 1); mbar_init(&raw_empty[s], 1); }
        for (int b = 0; b < 2; ++b) {
            mbar_init(&w_ready[b], 1); mbar_init(&w_free[b], 1);
            mbar_init(&tmem_full[b], 1); mbar_init(&tmem_empty[b], kEpiWarps);
        }
        for (int s = 0; s < kDescRing; ++s) { mbar_init(&d_ready[s], 1); mbar_init(&d_free[s], kDescReaders); }
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

#ifdef QR_PROF
    long long prof[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    const long long prof_t0 = clock64();
#define PW(cls, bar, par) do { const long long t_ = clock64(); mbar_wait_quiet(bar, par); prof[cls] += clock64() - t_; } while (0)
#else
#ifdef QR_QUIET
#define PW(cls, bar, par) mbar_wait_quiet(bar, par)
#else
#define PW(cls, bar, par) mbar_wait(bar, par)
#endif
#endif
    // every role walks the same sequence of descriptors h = 0, 1, ...; the scheduler warp publishes them, and a ring slot is
    // reused only after every consumer warp is through with that half tile (desc_done: what it read from the slot has
    // long been used by then -- an mbarrier arrive does not wait for the warp's outstanding shared-memory loads)
    auto desc_done = [&](int h) {
        __syncwarp();
        if (lane == 0) mbar_arrive(&d_free[h % kDescRing]);
    };
    auto wait_desc = [&](int h) -> const MmaDesc* {
        PW(0, &d_ready[h % kDescRing], (uint32_t)((h / kDescRing) & 1));
        return &desc[h % kDescRing];
    };

    if (warp < kEpiWarps) {
        // ================================================= epilogue =================================================
        // thread = pixel m = 32 warp + lane of the half tile (row-major 16 x 8: the warp owns image rows 2 warp, 2 warp + 1):
        // TMEM lane m, 256 columns = channels.  32 channels at a time: two tcgen05.ld.x16 -> eight 16-byte st.shared into
        // a [32 px][128 B] tile in the TMA 128-byte swizzle (chunk j of row r lands in chunk j ^ (r & 7): conflict free)
        // -> one TMA tensor store of the box {32 channels, 16 x, 2 y}; pixels outside the image are clipped by the TMA.
        unsigned char* my_out = smem + MmaSmem::out + warp * kOutBufs * kOutTile;
        const uint32_t row_off = (uint32_t)lane * 128u;
        const uint32_t sw = (uint32_t)(lane & 7);
        auto ld16 = [&](uint32_t taddr, uint32_t (&r)[16]) {
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                         : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                           "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                         : "r"(taddr));
        };
        int unit = 0, nbuf = 0;
        for (int h = 0;; ++h) {
            const MmaDesc* d = wait_desc(h);
            if (d->end) break;
            const int ht = d->ht;
            const int tile = ht >> 1;
            const int x0 = (tile % p.cam.tiles_x) * kTile, y0 = (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8 + 2 * warp;
            for (int c = 0; c < nunits; ++c, ++unit) {
                const int buf = unit & 1;
                PW(1, &tmem_full[buf], (unit >> 1) & 1);
                tc_fence_after();
                const uint32_t t0 = tmem_base + ((uint32_t)(warp * 32) << 16) + (uint32_t)(buf * kUnitN);
#pragma unroll 1
                for (int ch = 0; ch < kUnitN / 32; ++ch, ++nbuf) {
                    uint32_t ra[16], rb[16];
                    ld16(t0 + ch * 32, ra);
                    ld16(t0 + ch * 32 + 16, rb);
                    unsigned char* tile_s = my_out + (nbuf % kOutBufs) * kOutTile;
                    // the TMA store that read this staging tile kOutBufs stores ago must be through with it
                    if (lane == 0) bulk_wait_read<kOutBufs - 1>();
                    __syncwarp();
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    if (ch == kUnitN / 32 - 1) {        // every tcgen05.ld of this accumulator has completed
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(&tmem_empty[buf]);
                    }
                    unsigned char* rowp = tile_s + row_off;
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        *reinterpret_cast<uint4*>(rowp + (((uint32_t)j ^ sw) << 4)) = make_uint4(ra[4 * j], ra[4 * j + 1], ra[4 * j + 2], ra[4 * j + 3]);
                        *reinterpret_cast<uint4*>(rowp + (((uint32_t)(j + 4) ^ sw) << 4)) = make_uint4(rb[4 * j], rb[4 * j + 1], rb[4 * j + 2], rb[4 * j + 3]);
                    }
                    fence_async_smem();
                    __syncwarp();
                    if (lane == 0) {
                        tma_store_3d(&out_tmap, tile_s, c * kUnitN + ch * 32, x0, y0);
                        bulk_commit();
                    }
                }
            }
            desc_done(h);
        }
        if (lane == 0) bulk_wait<0>();
    } else if (warp == kMmaWarp) {
        // ================================================= MMA issuer ===============================================
        // The whole warp runs the loop in uniform control flow (descriptors stay in uniform registers); one elected
        // lane issues the tcgen05 instructions.
        // M = 128, N = 128, fp32 accumulate, A (tensor memory, K-major) and B (shared memory, MN-major) tf32
        const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | (1u << 16) | ((uint32_t)(kUnitN >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
        const uint32_t st0 = s32(stage_base);
        int unit = 0, wi = 0, st = 0;                      // wi: W instances consumed so far; instance i is in buffer i & 1
        for (int h = 0;; ++h) {
            const MmaDesc* d = wait_desc(h);
            if (d->end) break;
            const int U = d->U;
            const int rounds = rounds_of(U);
            const bool reuse = rounds <= 2;                // both W instances stay resident for every unit of the half tile
            const int wi0 = wi;
            for (int c = 0; c < nunits; ++c, ++unit) {
                const int buf = unit & 1;
                PW(1, &tmem_empty[buf], ((unit >> 1) & 1) ^ 1);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + (uint32_t)(buf * kUnitN);
                for (int r = 0; r < rounds; ++r) {
                    const int inst = reuse ? wi0 + r : wi++;
                    if (!reuse || c == 0) { PW(2, &w_ready[inst & 1], (inst >> 1) & 1); tc_fence_after(); }
                    const uint32_t a_hi = tmem_base + (uint32_t)(kTmemW + (inst & 1) * 2 * kWCols), a_lo = a_hi + kWCols;
                    const int nk = ksteps_of(cols_of(U, r));
                    for (int j = 0; j < nk; ++j, ++st) {
                        const int s = st % kStages;
                        PW(3, &full[s], (st / kStages) & 1);
                        tc_fence_after();
                        const uint32_t b_hi = st0 + s * kStageBytes, b_lo = b_hi + kStageHalf;
                        const uint64_t db_hi = umma_desc(b_hi, 1024, 512, 1);
                        const uint64_t db_lo = umma_desc(b_lo, 1024, 512, 1);
                        if (elect_one()) {
                            umma_tf32_ts(d_tmem, a_hi + j * kStageRows, db_hi, idesc, (r | j) != 0);
                            umma_tf32_ts(d_tmem, a_lo + j * kStageRows, db_hi, idesc, true);
                            if (!f16) umma_tf32_ts(d_tmem, a_hi + j * kStageRows, db_lo, idesc, true);
                            umma_commit(&empty[s]);
                        }
                        __syncwarp();
                    }
                    if (!reuse || c == nunits - 1) {                     // last use of this W instance
                        if (elect_one()) umma_commit(&w_free[inst & 1]);
                        __syncwarp();
                    }
                }
                if (elect_one()) umma_commit(&tmem_full[buf]);
                __syncwarp();
            }
            if (reuse) wi = wi0 + rounds;
            desc_done(h);
        }
    } else if (warp >= kLoadWarp && warp < kLoadWarp + kLoadWarps) {
        // ================================================= loader ===================================================
        // lane k < 8 copies union row 8 j + k of every stage: 512 B (128 channels) per bulk copy, kRawStages ahead.  The
        // union's ids come from the walk's lists in global memory (L2 loads: the walk may still be running elsewhere).
        unsigned char* raw_base = smem + MmaSmem::raw;
        int st = 0;
        for (int h = 0;; ++h) {
            const MmaDesc* d = wait_desc(h);
            if (d->end) break;
            const int U = d->U;
            const int32_t* uid = p.sl.uid + (size_t)d->ht * p.sl.ucap;
            const int32_t* uid_h = uid_s + (h % kDescRing) * kUidS;
            int32_t my_ids[kUidS / 32];                    // the shared ids of this half tile, lane-strided, copied out
#pragma unroll
            for (int q = 0; q < kUidS / 32; ++q) my_ids[q] = q * 32 + lane < U ? uid_h[q * 32 + lane] : 0;
            const int rounds = rounds_of(U);
            for (int c = 0; c < nunits; ++c) {
                for (int r = 0; r < rounds; ++r) {
                    const int ncols = cols_of(U, r);
                    const int nk = ksteps_of(ncols);
                    for (int j = 0; j < nk; ++j, ++st) {
                        if (st % kLoadWarps != warp - kLoadWarp) continue;
                        const int s = st % kRawStages;
                        const int rows = max(0, min(kStageRows, ncols - j * kStageRows));
                        int32_t id = 0;
                        {   // union id of row `lane` of the stage: from the copied ids (a shuffle), else from the lists
                            const int col = r * kWCols + j * kStageRows + (lane & 7);
                            int32_t v = 0;
#pragma unroll
                            for (int q = 0; q < kUidS / 32; ++q) {
                                const int32_t t = __shfl_sync(0xffffffffu, my_ids[q], col & 31);
                                if ((col >> 5) == q) v = t;
                            }
                            if (lane < rows) id = col < kUidS ? v : __ldcg(uid + col);
                        }
                        // lane g < 2 gathers rows 4 g .. 4 g + 3 with one instruction; rows past the union repeat a valid id
                        // (the converters zero them)
                        const int ngrp = (rows + 3) >> 2;
                        int ids4[4];
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const int src = min(4 * (lane & 1) + k, max(rows - 1, 0));
                            ids4[k] = __shfl_sync(0xffffffffu, id, src);
                        }
                        PW(1, &raw_empty[s], ((st / kRawStages) & 1) ^ 1);
                        if (lane == 0) {
                            if (ngrp > 0) mbar_arrive_expect_tx(&raw_full[s], (uint32_t)(ngrp * 4 * raw_row));
                            else mbar_arrive(&raw_full[s]);
                        }
                        __syncwarp();
                        if (lane < ngrp)
                            tma_gather4(raw_base + s * kRawBytes + lane * 4 * raw_row, &feat_tmap, c * kUnitN,
                                        ids4[0], ids4[1], ids4[2], ids4[3], &raw_full[s]);
                    }
                }
            }
            desc_done(h);
        }
    } else if (warp == kSchedWarp) {
        // ================================================= scheduler ================================================
        // runs up to kDescRing half tiles ahead of the pipeline: claims the next half tile inside the image (global ticket,
        // index order = the order the walk produces them), waits for its release flag, and publishes {half tile, list
        // lengths, union size} plus the first kUidS union ids in shared memory.  Every global round trip of the hand-over
        // (ticket, flag, header, ids) happens here, off the critical path of the builders and loaders.
        for (int h = 0;; ++h) {
            const int slot = h % kDescRing;
            PW(1, &d_free[slot], (uint32_t)(((h / kDescRing) & 1) ^ 1));
            MmaDesc* d = &desc[slot];
            int ht = 0;
            if (lane == 0) {
                while (true) {
                    ht = atomicAdd(p.sl.ctrl + 1, 1);
                    if (ht >= num_half) break;
                    const int y0 = ((ht >> 1) / p.cam.tiles_x) * kTile + (ht & 1) * 8;
                    if (y0 < p.cam.height) break;
                }
                if (ht < num_half) {
                    const int32_t* flag = p.sl.flags + ht;
#ifdef QR_PROF
                    const long long tf_ = clock64();
#endif
                    while (ld_acquire(flag) == 0) __nanosleep(500);
#ifdef QR_LAG
                    { const int32_t* f2 = p.sl.flags + min(ht + QR_LAG, num_half - 1); while (ld_acquire(f2) == 0) __nanosleep(500); }
#endif
#ifdef QR_PROF
                    prof[2] += clock64() - tf_;
#endif
                }
            }
            ht = __shfl_sync(0xffffffffu, ht, 0);            // (also orders the other lanes' loads after the acquire)
            const bool end = ht >= num_half;
            int U = 0;
            if (!end) {
                const int32_t* hd = p.sl.hdr + (size_t)ht * kHdrWords;
                const int32_t v = lane < 5 ? __ldcg(hd + lane) : 0;
                U = __shfl_sync(0xffffffffu, v, 4);
                if (lane < 4) (&d->n0)[lane] = v;
                const int32_t* uid = p.sl.uid + (size_t)ht * p.sl.ucap;
#pragma unroll
                for (int q = 0; q < kUidS / 32; ++q)
                    if (q * 32 + lane < U) uid_s[slot * kUidS + q * 32 + lane] = __ldcg(uid + q * 32 + lane);
            }
            if (lane == 0) { d->ht = ht; d->U = U; d->end = end ? 1 : 0; }
            __threadfence_block();
            __syncwarp();
            if (lane == 0) mbar_arrive(&d_ready[slot]);
            if (end) break;
        }
    } else if (warp >= kFirstConv && warp < kFirstBuild) {
        // ================================================= converters ===============================================
        // converter warp pw owns the stages st with st % 3 == pw (all 8 union rows of the stage): ld.shared of the raw rows ->
        // hi / lo -> st.shared in the MN-major SWIZZLE_128B_BASE32B layout.  One warp per stage, three stages in flight:
        // with the rows of ONE stage spread over the warps every hand-over latency (barrier wake-up, ld.shared,
        // fence.proxy.async) was paid 24 times in series per half tile and the MMA warp starved.
        const int pw = warp - kFirstConv;                 // 0..2
        const unsigned char* raw_base = smem + MmaSmem::raw;
        // byte offset of this lane's 16 bytes (channels 4 lane .. 4 lane + 3) inside a stage half, row q of the stage
        auto lane_off = [&](int q) -> uint32_t {
            return (uint32_t)((lane >> 3) * 1024 + (q >> 2) * 512 + (q & 3) * 128 + ((((lane & 7) >> 1) ^ (q & 3)) * 32) + (lane & 1) * 16);
        };
        int st = 0;
        for (int h = 0;; ++h) {
            const MmaDesc* d = wait_desc(h);
            if (d->end) break;
            const int U = d->U;
            const int rounds = rounds_of(U);
            for (int c = 0; c < nunits; ++c) {
                for (int r = 0; r < rounds; ++r) {
                    const int ncols = cols_of(U, r);
                    const int nk = ksteps_of(ncols);
                    for (int j = 0; j < nk; ++j, ++st) {
                        if (st % kConvWarps != pw) continue;
                        const int sr = st % kRawStages;
                        PW(1, &raw_full[sr], (st / kRawStages) & 1);
                        const int rows = max(0, min(kStageRows, ncols - j * kStageRows));
                        float4 a[kStageRows];
#pragma unroll
                        for (int q = 0; q < kStageRows; ++q) {
                            a[q] = make_float4(0.f, 0.f, 0.f, 0.f);
                            if (q < rows) {
                                if (f16) {
                                    const uint2 h = *reinterpret_cast<const uint2*>(raw_base + sr * kRawBytes + q * raw_row + lane * 8);
                                    const float2 f0 = __half22float2(*reinterpret_cast<const __half2*>(&h.x));
                                    const float2 f1 = __half22float2(*reinterpret_cast<const __half2*>(&h.y));
                                    a[q] = make_float4(f0.x, f0.y, f1.x, f1.y);
                                } else {
                                    a[q] = *reinterpret_cast<const float4*>(raw_base + sr * kRawBytes + q * kRawRow + lane * 16);
                                }
                            }
                        }
                        const int s = st % kStages;
                        PW(2, &empty[s], ((st / kStages) & 1) ^ 1);
                        unsigned char* stg = stage_base + s * kStageBytes;
#pragma unroll
                        for (int q = 0; q < kStageRows; ++q) {
                            unsigned char* hi = stg + lane_off(q);
                            const float4 v = a[q];
                            const float4 hv = make_float4(tf32_hi(v.x), tf32_hi(v.y), tf32_hi(v.z), tf32_hi(v.w));
                            *reinterpret_cast<float4*>(hi) = hv;
                            if (!f16)
                                *reinterpret_cast<float4*>(hi + kStageHalf) =
                                    make_float4(__fsub_rn(v.x, hv.x), __fsub_rn(v.y, hv.y), __fsub_rn(v.z, hv.z), __fsub_rn(v.w, hv.w));
                        }
                        fence_async_smem();
                        __syncwarp();
                        // the raw slot is released only now: the loads above have provably completed (their values were
                        // stored), so the loader's next TMA write cannot overtake a read still queued in the LSU
                        if (lane == 0) { mbar_arrive(&raw_empty[sr]); mbar_arrive(&full[s]); }
                    }
                }
            }
            desc_done(h);
        }
    } else if (warp >= kFirstBuild) {
        // ================================================= builders =================================================
        const int ptid = (warp & 3) * 32 + lane;          // 0..127 = pixel of the half tile = TMEM lane (a warp reaches the lane quarter warp % 4)
        auto prod_sync = [&]() { named_sync<1, kBuildThreads>(); };
        float* ws = reinterpret_cast<float*>(smem + MmaSmem::w);
        auto st8 = [&](uint32_t taddr, const uint32_t (&r)[8]) {
            asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                         ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]) : "memory");
        };
        const uint32_t lane_base = ((uint32_t)((warp & 3) * 32)) << 16;
        int wi = 0;                                       // W instances built so far; instance i goes to buffer i & 1
        // builder warp q scatters list q (the walk's warp q wrote it).  The first kEbuf entries of the list are staged in
        // shared memory by cp.async while the PREVIOUS instance is stored to tensor memory, so the scatter never waits for
        // an L2 round trip; the rare longer lists read their tail straight from global memory.
        const int bq = warp - kFirstBuild;
        uint2* ebuf = reinterpret_cast<uint2*>(smem + MmaSmem::ebuf) + bq * kEbuf;
        struct HT { int ht, U, n, end; };
        auto read_desc = [&](int h) -> HT {
            const MmaDesc* d = wait_desc(h);
            HT t;
            t.end = d->end; t.ht = d->ht; t.U = d->U;
            t.n = (&d->n0)[bq];
            return t;
        };
        auto stage_entries = [&](const HT& t) {             // 16 bytes = 2 entries per cp.async
            const uint2* src = p.sl.ent + ((size_t)t.ht * kSelLists + bq) * p.sl.qcap;
            const int n2 = (min(t.n, kEbuf) + 1) >> 1;
            for (int i = lane; i < n2; i += 32)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s32(ebuf + 2 * i)), "l"(src + 2 * i) : "memory");
            asm volatile("cp.async.commit_group;" ::: "memory");
        };
        HT cur = read_desc(0);
        if (!cur.end) stage_entries(cur);
        for (int h = 0; !cur.end; ++h) {
            const int rounds = rounds_of(cur.U);
            const int ninst = rounds <= 2 ? rounds : rounds * nunits;      // (the MMA warp derives the same sequence)
            const uint2* tail = p.sl.ent + ((size_t)cur.ht * kSelLists + bq) * p.sl.qcap;
            HT nxt = cur;
            for (int ii = 0; ii < ninst; ++ii, ++wi) {
                const int r = ii % rounds;
                // ---------------- build W for columns [64 r, 64 r + 64) ----------------
#ifdef QR_PROF
                const long long tb0_ = clock64();
#endif
                {
                    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
                    float4* wz = reinterpret_cast<float4*>(ws);
                    for (int i = ptid; i < kWsBytes / 16; i += kBuildThreads) wz[i] = z;
                }
                asm volatile("cp.async.wait_all;" ::: "memory");     // this warp's staged entries have landed
                prod_sync();
                const int c_lo = r * kWCols;
                for (int i = lane; i < min(cur.n, kEbuf); i += 32) {
                    const uint2 e = ebuf[i];
                    const int cl = sel_col(e.y) - c_lo;
                    if (cl >= 0 && cl < kWCols) ws[sel_pixel(e.y) * kWsRow + cl] = __uint_as_float(e.x);
                }
                // the tail of a long list (rare for Q-Render; the rule for the dense comparator's lists, ~60 entries per pixel)
                // comes straight from global memory, eight loads per lane in flight
                for (int i0 = kEbuf + lane; i0 < cur.n; i0 += 32 * 8) {
                    uint2 e[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u) e[u] = i0 + 32 * u < cur.n ? __ldcg(tail + i0 + 32 * u) : make_uint2(0u, 0xFFFFFFFFu);
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const int cl = sel_col(e[u].y) - c_lo;            // padding: column 2^17 - 1, never in range
                        if (cl >= 0 && cl < kWCols) ws[sel_pixel(e[u].y) * kWsRow + cl] = __uint_as_float(e[u].x);
                    }
                }
                prod_sync();
#ifdef QR_PROF
                const long long tb1_ = clock64();
                prof[2] += tb1_ - tb0_;
#endif
                // the scratch tile is complete; after the last instance of this half tile the staging buffer is free:
                // request the next half tile's entries now, they land during the tensor-memory phase below
                if (ii + 1 == ninst) { nxt = read_desc(h + 1); if (!nxt.end) stage_entries(nxt); }
                // thread = pixel: its row of 64 weights -> tensor memory, hi (the raw value: kind::tf32 reads its top 19
                // bits) and lo = w - trunc(w); the buffer is free once the MMAs of the instance two before have retired
                PW(1, &w_free[wi & 1], ((wi >> 1) & 1) ^ 1);
                tc_fence_after();
                const uint32_t t_hi = tmem_base + lane_base + (uint32_t)(kTmemW + (wi & 1) * 2 * kWCols);
                const float4* row = reinterpret_cast<const float4*>(ws + ptid * kWsRow);
#pragma unroll 2
                for (int q = 0; q < kWCols / 8; ++q) {
                    const float4 v0 = row[2 * q], v1 = row[2 * q + 1];
                    const float f[8] = { v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w };
                    uint32_t hi[8], lo[8];
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        hi[i] = __float_as_uint(f[i]);
                        lo[i] = __float_as_uint(__fsub_rn(f[i], tf32_hi(f[i])));
                    }
                    st8(t_hi + q * 8, hi);
                    st8(t_hi + kWCols + q * 8, lo);
                }
                asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                tc_fence_before();
                prod_sync();                                 // every row is in tensor memory; the scratch tile is free again
#ifdef QR_PROF
                prof[3] += clock64() - tb1_;
#endif
                if (ptid == 0) mbar_arrive(&w_ready[wi & 1]);
            }
            desc_done(h);                                    // (the fields of descriptor h + 1 were copied out after a barrier)
            cur = nxt;
        }
    }

#ifdef QR_PROF
    if (lane == 0) {    // role = warp group; ctrl[16 + 8 role + class] in units of 1024 cycles, class 7 = total
        const int role = warp < 4 ? 0 : (warp == 4 ? 1 : (warp < 8 ? 2 : (warp == 8 ? 5 : (warp < 12 ? 3 : 4))));
        prof[7] = clock64() - prof_t0;
        for (int c = 0; c < 8; ++c) atomicAdd(p.sl.ctrl + 16 + 8 * role + c, (int)(prof[c] >> 10));
    }
#endif
    tc_fence_before();
    __syncthreads();
    if (tid == 0) stamp_time(p.sl.ctrl, 3, false);
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
}

bool blend_mma_supported(int32_t D, qr_dtype feat_dtype)
{
    return tc_channels_supported(D) && (feat_dtype == QR_F32 || (feat_dtype == QR_F16 && D % 8 == 0));
}

int launch_blend_mma(const BlendParams& p, cudaStream_t st, bool pdl)
{
    // out_map [H][W][D] fp32 as a 3-D tensor (D, W, H); box = 32 channels x 16 pixels x 2 rows, 128-byte swizzle
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return fail(QR_ERR_CUDA, "qr_forward: cuTensorMapEncodeTiled is not available from the driver");
    CUtensorMap tmap;
    const cuuint64_t dims[3] = { (cuuint64_t)p.D, (cuuint64_t)p.cam.width, (cuuint64_t)p.cam.height };
    const cuuint64_t strides[2] = { (cuuint64_t)p.D * 4, (cuuint64_t)p.D * 4 * (cuuint64_t)p.cam.width };
    const cuuint32_t box[3] = { 32, 16, 2 };
    const cuuint32_t estr[3] = { 1, 1, 1 };
    const CUresult cr = enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, p.out_map, dims, strides, box, estr,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) return fail(QR_ERR_CUDA, "qr_forward: cuTensorMapEncodeTiled failed (%d)", (int)cr);
    // features [N][D] fp32 as a 2-D tensor (D, N) for tile::gather4: box = 128 channels x 1 row, no swizzle
    CUtensorMap fmap;
    {
        // (qr_forward is not told N: the row bound is left open, ids come from the caller's own intersection lists)
        const cuuint64_t fdims[2] = { (cuuint64_t)p.D, (cuuint64_t)0x7fffffff };
        const cuuint64_t fstr[1] = { (cuuint64_t)p.D * (p.feat_f16 ? 2 : 4) };
        const cuuint32_t fbox[2] = { (cuuint32_t)kUnitN, 1 };
        const cuuint32_t fes[2] = { 1, 1 };
        const CUresult fr = enc(&fmap, p.feat_f16 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(p.features), fdims, fstr, fbox, fes,
                                CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (fr != CUDA_SUCCESS) return fail(QR_ERR_CUDA, "qr_forward: cuTensorMapEncodeTiled (features) failed (%d)", (int)fr);
    }
    const int sms = sm_count();
    const unsigned grid = (unsigned)min(sms, p.num_tiles * 2);
    QR_CUDA_OK(cudaFuncSetAttribute(blend_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, MmaSmem::total));
    // programmatic dependent launch: the kernel does not wait for walk2_kernel to finish (it never calls
    // griddepcontrol.wait); it starts once every walk CTA has started and synchronises per half tile through the
    // release flags.  If the two kernels are serialised (a profiler, a full GPU) the flags are simply all set.
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(kMmaThreads); cfg.dynamicSmemBytes = MmaSmem::total; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = (pdl && !getenv("QR_NO_PDL")) ? 1 : 0;     // QR_NO_PDL: serialise the two kernels (profiling)
    QR_CUDA_OK(cudaLaunchKernelEx(&cfg, blend_mma_kernel, p, tmap, fmap));
    QR_LAUNCH_OK("blend_mma_kernel");
    return QR_OK;
}

}  // namespace qr

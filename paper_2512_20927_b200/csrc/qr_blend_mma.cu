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
// One persistent CTA per SM, 16 warps (512 threads, <= 64 registers: the kernel is meant to share its SM with CTAs of
// walk2_kernel, which it follows by programmatic dependent launch), roles by warp, no role ever waits at a block barrier:
//   warps 0..3    epilogue: tcgen05.ld of the accumulator (thread = pixel), st.shared into a 128-byte-swizzled staging
//                 tile, one TMA tensor store per (32 pixels x 32 channels): the map leaves the SM as whole 128-byte lines
//   warp  4       MMA issue: warp-uniform loop, one elected lane issues tcgen05.mma (M = 128 pixels, N = 256 channels,
//                 K = 8 union rows per instruction) and tcgen05.commit
//   warp  5       loader: one bulk async copy (TMA) per feature row half (1 KB) into a raw ring, ahead of use
//   warps 8..11   converters: ld.shared of a raw row -> hi/lo split -> st.shared in the MN-major
//                 SWIZZLE_128B_BASE32B layout tf32 needs for a row-major (channel-contiguous) B operand
//   warps 12..15  builders: claim the next half tile (global ticket, same order as the walk), wait for its ready flag,
//                 publish its descriptor to the other roles, then build W (K-major, no swizzle; hi and lo) from the
//                 entry lists: thread = entry, loads issued before the wait on the buffer
// Work unit = (half tile, 256-channel half): two 256-column accumulators in TMEM, so the MMAs of unit i+1 overlap the
// epilogue of unit i.  A half tile whose union exceeds 64 columns is processed in rounds of 64 columns.
#include <cuda.h>

#include "qr_async.cuh"
#include "qr_blend.cuh"

namespace qr {

using namespace aq;

constexpr int kEpiWarps = 4;
constexpr int kMmaWarp = 4;
constexpr int kLoadWarp = 5;
constexpr int kFirstConv = 8;
constexpr int kConvWarps = 4;                             // two union rows of every stage each
constexpr int kFirstBuild = 12;
constexpr int kBuildWarps = 4;
constexpr int kMmaThreads = (kFirstBuild + kBuildWarps) * 32;   // 512
constexpr int kBuildThreads = kBuildWarps * 32;
constexpr int kWCols = 64;                                // union columns per round
constexpr int kUnitN = 256;                               // channels per work unit
constexpr int kStageRows = 8;                             // union rows per stage = one tf32 K step
constexpr int kStages = 2;
constexpr int kRawStages = 4;
constexpr int kRawRow = kUnitN * 4;                       // 1 KB: one feature row half
constexpr int kRawBytes = kStageRows * kRawRow;           // 8 KB per raw stage
constexpr int kWBytes = 128 * kWCols * 4;                 // 32 KB (hi or lo)
constexpr int kStageHalf = kStageRows * kUnitN * 4;       // 8 KB (hi or lo)
constexpr int kStageBytes = 2 * kStageHalf;
constexpr int kOutBufs = 3;                               // staging tiles per epilogue warp
constexpr int kOutTile = 32 * 128;                        // 32 pixels x 32 channels fp32
constexpr int kDescRing = 4;
constexpr int kEntRegs = 8;                               // entries a builder thread holds in flight

struct MmaDesc { int32_t ht, U, n0, n1, n2, n3, end, pad; };

struct MmaSmem {
    static constexpr int w = 0;                                           // [hi, lo]
    static constexpr int stages = 2 * kWBytes;
    static constexpr int raw = stages + kStages * kStageBytes;
    static constexpr int out = raw + kRawStages * kRawBytes;              // [4 warps][kOutBufs] staging tiles, 1 KB aligned
    static constexpr int desc = out + kEpiWarps * kOutBufs * kOutTile;
    static constexpr int bars = desc + kDescRing * (int)sizeof(MmaDesc);
    static constexpr int n_bars = 2 * kStages + 2 * kRawStages + 2 + 4 + kDescRing;
    static constexpr int tmem = bars + n_bars * 8;
    static constexpr int total = tmem + 16;
};

__device__ __forceinline__ void umma_commit(uint64_t* bar)     // arrives when every MMA issued so far by this thread is done
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(s32(bar)) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// shared-memory matrix descriptor (sm_100): start >> 4 | LBO >> 4 << 16 | SBO >> 4 << 32 | version 1 << 46 | layout << 61
__device__ __forceinline__ uint64_t umma_desc(uint32_t addr, uint32_t lbo, uint32_t sbo, uint32_t layout)
{
    return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)((lbo >> 4) & 0x3FFF) << 16) |
           ((uint64_t)((sbo >> 4) & 0x3FFF) << 32) | ((uint64_t)1 << 46) | ((uint64_t)layout << 61);
}
__device__ __forceinline__ void umma_tf32(uint32_t d_tmem, uint64_t a, uint64_t b, uint32_t idesc, bool accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(a), "l"(b), "r"(idesc), "r"((uint32_t)accumulate) : "memory");
}
__device__ __forceinline__ bool elect_one()     // one lane of a converged warp, always the same one
{
    uint32_t pred;
    asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.u32 %0, 1, 0, P;\n\t}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ float tf32_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xFFFFE000u); }
__device__ __forceinline__ int32_t ld_acquire(const int32_t* p)
{
    int32_t v;
    asm volatile("ld.acquire.gpu.global.b32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* map, const void* src, int c0, int x, int y)
{
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];"
                 ::"l"(reinterpret_cast<uint64_t>(map)), "r"(s32(src)), "r"(c0), "r"(x), "r"(y) : "memory");
}

// byte offset of W[m][c] in the K-major, non-swizzled canonical layout: core matrix = 8 pixels x 4 columns (128 B);
// column chunks 128 B apart (LBO), 8-pixel groups 2 KB apart (SBO)
__device__ __forceinline__ uint32_t w_off(int m, int c)
{
    return (uint32_t)((m >> 3) * (kWCols / 4 * 128) + (c >> 2) * 128 + (m & 7) * 16 + (c & 3) * 4);
}

// rounds / K steps of a half tile: every role derives them from the union size
__device__ __forceinline__ int rounds_of(int U) { return U <= kWCols ? 1 : (U + kWCols - 1) / kWCols; }
__device__ __forceinline__ int cols_of(int U, int r) { return max(0, min(kWCols, U - r * kWCols)); }
__device__ __forceinline__ int ksteps_of(int ncols) { return max(1, (ncols + kStageRows - 1) / kStageRows); }

__global__ void __launch_bounds__(kMmaThreads, 2)       // "2" only caps the registers at 64; shared memory allows one CTA
blend_mma_kernel(const BlendParams p, const __grid_constant__ CUtensorMap out_tmap)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char* stage_base = smem + MmaSmem::stages;
    MmaDesc* desc = reinterpret_cast<MmaDesc*>(smem + MmaSmem::desc);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + MmaSmem::bars);
    uint64_t* full = bars;                       // [kStages] converters -> MMA (4 warp arrivals)
    uint64_t* empty = bars + kStages;            // [kStages] MMA -> converters (tcgen05.commit)
    uint64_t* raw_full = bars + 2 * kStages;     // [kRawStages] loader (TMA complete_tx) -> converters
    uint64_t* raw_empty = raw_full + kRawStages; // [kRawStages] converters -> loader (4 warp arrivals)
    uint64_t* w_ready = raw_empty + kRawStages;  // builders -> MMA
    uint64_t* w_free = w_ready + 1;              // MMA -> builders (tcgen05.commit)
    uint64_t* tmem_full = w_free + 1;            // [2] MMA -> epilogue (tcgen05.commit)
    uint64_t* tmem_empty = tmem_full + 2;        // [2] epilogue -> MMA (4 warp arrivals)
    uint64_t* d_ready = tmem_empty + 2;          // [kDescRing] builders -> everybody: descriptor h is published
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + MmaSmem::tmem);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int D = p.D;
    const int nunits = D / kUnitN;
    const int num_half = p.num_tiles * 2;

    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) { mbar_init(&full[s], kConvWarps); mbar_init(&empty[s], 1); }
        for (int s = 0; s < kRawStages; ++s) { mbar_init(&raw_full[s], 1); mbar_init(&raw_empty[s], kConvWarps); }
        mbar_init(w_ready, 1); mbar_init(w_free, 1);
        for (int b = 0; b < 2; ++b) { mbar_init(&tmem_full[b], 1); mbar_init(&tmem_empty[b], kEpiWarps); }
        for (int s = 0; s < kDescRing; ++s) mbar_init(&d_ready[s], 1);
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

    // every role walks the same sequence of descriptors h = 0, 1, ...; the builders publish them
    auto wait_desc = [&](int h) -> const MmaDesc* {
        mbar_wait(&d_ready[h % kDescRing], (uint32_t)((h / kDescRing) & 1));
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
                mbar_wait(&tmem_full[buf], (unit >> 1) & 1);
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
        }
        if (lane == 0) bulk_wait<0>();
    } else if (warp == kMmaWarp) {
        // ================================================= MMA issuer ===============================================
        // The whole warp runs the loop in uniform control flow (descriptors stay in uniform registers); one elected
        // lane issues the tcgen05 instructions.
        // M = 128, N = 256, fp32 accumulate, A and B tf32, A K-major, B MN-major
        const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | (1u << 16) | ((uint32_t)(kUnitN >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
        const uint32_t a_hi = s32(smem + MmaSmem::w), a_lo = a_hi + kWBytes, st0 = s32(stage_base);
        int unit = 0, wi = 0, st = 0;                      // wi: W instances consumed so far
        for (int h = 0;; ++h) {
            const MmaDesc* d = wait_desc(h);
            if (d->end) break;
            const int U = d->U;
            const int rounds = rounds_of(U);
            for (int c = 0; c < nunits; ++c, ++unit) {
                const int buf = unit & 1;
                mbar_wait(&tmem_empty[buf], ((unit >> 1) & 1) ^ 1);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + (uint32_t)(buf * kUnitN);
                for (int r = 0; r < rounds; ++r) {
                    if (c == 0 || rounds > 1) { mbar_wait(w_ready, wi & 1); ++wi; }
                    const int nk = ksteps_of(cols_of(U, r));
                    for (int j = 0; j < nk; ++j, ++st) {
                        const int s = st % kStages;
                        mbar_wait(&full[s], (st / kStages) & 1);
                        tc_fence_after();
                        const uint32_t b_hi = st0 + s * kStageBytes, b_lo = b_hi + kStageHalf;
                        const uint64_t da_hi = umma_desc(a_hi + j * 256, 128, kWCols / 4 * 128, 0);
                        const uint64_t da_lo = umma_desc(a_lo + j * 256, 128, kWCols / 4 * 128, 0);
                        const uint64_t db_hi = umma_desc(b_hi, 1024, 512, 1);
                        const uint64_t db_lo = umma_desc(b_lo, 1024, 512, 1);
                        if (elect_one()) {
                            umma_tf32(d_tmem, da_hi, db_hi, idesc, (r | j) != 0);
                            umma_tf32(d_tmem, da_lo, db_hi, idesc, true);
                            umma_tf32(d_tmem, da_hi, db_lo, idesc, true);
                            umma_commit(&empty[s]);
                        }
                        __syncwarp();
                    }
                    if (rounds > 1 || c == nunits - 1) {                 // last use of this W
                        if (elect_one()) umma_commit(w_free);
                        __syncwarp();
                    }
                }
                if (elect_one()) umma_commit(&tmem_full[buf]);
                __syncwarp();
            }
        }
    } else if (warp == kLoadWarp) {
        // ================================================= loader ===================================================
        // lane k < 8 copies union row 8 j + k of every stage: 1 KB (256 channels) per bulk copy, kRawStages ahead.  The
        // union's ids come from the walk's lists in global memory (L2 loads: the walk may still be running elsewhere).
        unsigned char* raw_base = smem + MmaSmem::raw;
        int st = 0;
        for (int h = 0;; ++h) {
            const MmaDesc* d = wait_desc(h);
            if (d->end) break;
            const int U = d->U;
            const int32_t* uid = p.sl.uid + (size_t)d->ht * p.sl.ucap;
            const int rounds = rounds_of(U);
            for (int c = 0; c < nunits; ++c) {
                for (int r = 0; r < rounds; ++r) {
                    const int ncols = cols_of(U, r);
                    const int nk = ksteps_of(ncols);
                    for (int j = 0; j < nk; ++j, ++st) {
                        const int s = st % kRawStages;
                        const int rows = max(0, min(kStageRows, ncols - j * kStageRows));
                        int32_t id = 0;
                        if (lane < rows) id = __ldcg(uid + r * kWCols + j * kStageRows + lane);
                        mbar_wait(&raw_empty[s], ((st / kRawStages) & 1) ^ 1);
                        if (lane == 0) {
                            if (rows > 0) mbar_arrive_expect_tx(&raw_full[s], (uint32_t)rows * kRawRow);
                            else mbar_arrive(&raw_full[s]);
                        }
                        __syncwarp();
                        if (lane < rows)
                            bulk_g2s(raw_base + s * kRawBytes + lane * kRawRow,
                                     static_cast<const float*>(p.features) + (int64_t)id * D + c * kUnitN, kRawRow, &raw_full[s]);
                    }
                }
            }
        }
    } else if (warp >= kFirstConv && warp < kFirstBuild) {
        // ================================================= converters ===============================================
        // warp pw splits union rows pw and pw + 4 of every stage: ld.shared of the raw row -> hi / lo -> st.shared in the
        // MN-major SWIZZLE_128B_BASE32B layout.
        const int pw = warp - kFirstConv;                 // 0..3
        const unsigned char* raw_base = smem + MmaSmem::raw;
        // byte offset of this lane's 16 bytes inside a stage half, row q of the stage: channels 4 lane .. 4 lane + 3 (+128)
        auto lane_off = [&](int q) -> uint32_t {
            return (uint32_t)((lane >> 3) * 1024 + (q >> 2) * 512 + (q & 3) * 128 + ((((lane & 7) >> 1) ^ (q & 3)) * 32) + (lane & 1) * 16);
        };
        const uint32_t off0 = lane_off(pw), off1 = lane_off(pw + 4);
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
                        const int sr = st % kRawStages;
                        mbar_wait(&raw_full[sr], (st / kRawStages) & 1);
                        float4 a[2][2];
#pragma unroll
                        for (int q = 0; q < 2; ++q) {
                            a[q][0] = a[q][1] = make_float4(0.f, 0.f, 0.f, 0.f);
                            if (j * kStageRows + pw + 4 * q < ncols) {
                                const unsigned char* rr = raw_base + sr * kRawBytes + (pw + 4 * q) * kRawRow + lane * 16;
                                a[q][0] = *reinterpret_cast<const float4*>(rr);
                                a[q][1] = *reinterpret_cast<const float4*>(rr + 512);
                            }
                        }
                        __syncwarp();
                        if (lane == 0) mbar_arrive(&raw_empty[sr]);          // the raw rows are in registers
                        const int s = st % kStages;
                        mbar_wait(&empty[s], ((st / kStages) & 1) ^ 1);
#pragma unroll
                        for (int q = 0; q < 2; ++q) {
                            unsigned char* hi = stage_base + s * kStageBytes + (q ? off1 : off0);
                            unsigned char* lo = hi + kStageHalf;
#pragma unroll
                            for (int t = 0; t < 2; ++t) {
                                const float4 v = a[q][t];
                                const float4 hv = make_float4(tf32_hi(v.x), tf32_hi(v.y), tf32_hi(v.z), tf32_hi(v.w));
                                *reinterpret_cast<float4*>(hi + t * 4 * 1024) = hv;
                                *reinterpret_cast<float4*>(lo + t * 4 * 1024) =
                                    make_float4(__fsub_rn(v.x, hv.x), __fsub_rn(v.y, hv.y), __fsub_rn(v.z, hv.z), __fsub_rn(v.w, hv.w));
                            }
                        }
                        fence_async_smem();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(&full[s]);
                    }
                }
            }
        }
    } else if (warp >= kFirstBuild) {
        // ================================================= builders =================================================
        const int ptid = tid - kFirstBuild * 32;          // 0..127
        auto prod_sync = [&]() { named_sync<1, kBuildThreads>(); };
        unsigned char* wbuf = smem + MmaSmem::w;
        int wi = 0;                                       // W instances built so far
        for (int h = 0;; ++h) {
            MmaDesc* d = &desc[h % kDescRing];
            if (ptid == 0) {
                // next half tile inside the image, in index order; its lists must be complete (the walk releases the flag)
                int ht;
                while (true) {
                    ht = atomicAdd(p.sl.ctrl + 1, 1);
                    if (ht >= num_half) break;
                    const int y0 = ((ht >> 1) / p.cam.tiles_x) * kTile + (ht & 1) * 8;
                    if (y0 < p.cam.height) break;
                }
                d->end = ht >= num_half ? 1 : 0;
                d->ht = ht;
                if (ht < num_half) {
                    const int32_t* flag = p.sl.flags + ht;
                    while (ld_acquire(flag) == 0) __nanosleep(200);
                    const int4 nq = __ldcg(reinterpret_cast<const int4*>(p.sl.hdr + (size_t)ht * kHdrWords));
                    d->n0 = nq.x; d->n1 = nq.y; d->n2 = nq.z; d->n3 = nq.w;
                    d->U = __ldcg(p.sl.hdr + (size_t)ht * kHdrWords + 4);
                }
                __threadfence_block();
                mbar_arrive(&d_ready[h % kDescRing]);
            }
            prod_sync();
            if (d->end) break;
            const int ht = d->ht, U = d->U;
            const int e1 = d->n0, e2 = e1 + d->n1, e3 = e2 + d->n2, total = e3 + d->n3;
            const uint2* ent = p.sl.ent + (size_t)ht * kSelLists * p.sl.qcap;
            auto ent_at = [&](int f) -> uint2 {            // flat index over the four lists
                const int q = (f >= e1) + (f >= e2) + (f >= e3);
                const int b = q == 0 ? 0 : (q == 1 ? e1 : (q == 2 ? e2 : e3));
                return __ldcg(ent + (size_t)q * p.sl.qcap + (f - b));
            };
            const int rounds = rounds_of(U);
            for (int c = 0; c < nunits; ++c) {
                for (int r = 0; r < rounds; ++r) {
                    if (c == 0 || rounds > 1) {
                        // ---------------- build W for columns [64 r, 64 r + 64) ----------------
                        uint2 e[kEntRegs];
#pragma unroll
                        for (int u = 0; u < kEntRegs; ++u) {
                            const int f = u * kBuildThreads + ptid;
                            e[u] = f < total ? ent_at(f) : make_uint2(0u, 0xFFFFFFFFu);
                        }
                        mbar_wait(w_free, (wi & 1) ^ 1);            // the MMAs that read the previous instance have retired
                        ++wi;
                        {
                            const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
                            float4* wz = reinterpret_cast<float4*>(wbuf);
                            for (int i = ptid; i < 2 * kWBytes / 16; i += kBuildThreads) wz[i] = z;
                        }
                        prod_sync();
                        for (int base = 0; base == 0 || base < total; base += kEntRegs * kBuildThreads) {
                            if (base > 0) {
#pragma unroll
                                for (int u = 0; u < kEntRegs; ++u) {
                                    const int f = base + u * kBuildThreads + ptid;
                                    e[u] = f < total ? ent_at(f) : make_uint2(0u, 0xFFFFFFFFu);
                                }
                            }
#pragma unroll
                            for (int u = 0; u < kEntRegs; ++u) {
                                const int cl = sel_col(e[u].y) - r * kWCols;       // padding entries have column 2^17 - 1
                                if (cl >= 0 && cl < kWCols) {
                                    const uint32_t off = w_off(sel_pixel(e[u].y), cl);
                                    const float w = __uint_as_float(e[u].x), hi = tf32_hi(w);
                                    *reinterpret_cast<float*>(wbuf + off) = hi;
                                    *reinterpret_cast<float*>(wbuf + kWBytes + off) = __fsub_rn(w, hi);
                                }
                            }
                        }
                        fence_async_smem();
                        prod_sync();
                        if (ptid == 0) mbar_arrive(w_ready);
                    }
                }
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
}

bool blend_mma_supported(int32_t D, qr_dtype feat_dtype) { return feat_dtype == QR_F32 && D >= kUnitN && D % kUnitN == 0; }

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* sym = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(sym);
    }
    return fn;
}

int launch_blend_mma(const BlendParams& p, cudaStream_t st)
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
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
        sms = 148;
    const unsigned grid = (unsigned)min(sms, p.num_tiles * 2);
    QR_CUDA_OK(cudaFuncSetAttribute(blend_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, MmaSmem::total));
    blend_mma_kernel<<<grid, kMmaThreads, MmaSmem::total, st>>>(p, tmap);
    QR_LAUNCH_OK("blend_mma_kernel");
    return QR_OK;
}

}  // namespace qr

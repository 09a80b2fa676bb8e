// qr_blend_mma.cu -- the O(KC) blend of qr_forward (Algorithm 1 lines 9 and 20) as a dense
// contraction on the 5th-generation tensor cores.
//
// Per 16x8-pixel half tile the blend is  out[128 px, D] = W[128 px, U] . F[U, D]  with U the union of the Gaussians
// selected by any of the 128 pixels (mean 47, 23 % dense at config 3) and W the sparse weights w^Q.  ncu showed the
// FFMA formulation of this product to be issue bound at 3x the time of its HBM traffic (profiles/README.md, r1_a),
// which is the evidence north_star asks for before putting it on tensor cores.
//
// Precision: kind::tf32 truncates its fp32 operands to 10 explicit mantissa bits (measured on B200), so both operands
// are split exactly, x = hi + lo with hi = x & 0xFFFFE000 and lo = x - hi, and three MMAs accumulate
// W_hi F_hi + W_lo F_hi + W_hi F_lo in fp32 (TMEM).  The dropped W_lo F_lo term and the truncation of the lo parts
// are <= 2^-21 relative per product, 40x below the fp32 tolerance of north_star (1e-4 relative).
//
// One persistent CTA per SM, 22 warps, roles by warp (no role ever waits at a block barrier):
//   warps 0..3    epilogue: tcgen05.ld of the accumulator (thread = pixel), x 1/(1 - T^Q), four 256-bit st.global per
//                 32 channels (a lane's 32 channels are 128 contiguous bytes of the map)
//   warp  4       MMA issue: warp-uniform loop, one elected lane issues tcgen05.mma (M = 128 pixels, N = 256 channels,
//                 K = 8 union rows per instruction) and tcgen05.commit
//   warp  5       loader: one bulk async copy (TMA) per feature row half (1 KB) into a raw ring, ahead of use
//   warps 6..13   converters: ld.shared of a raw row -> hi/lo split -> st.shared in the MN-major
//                 SWIZZLE_128B_BASE32B layout tf32 needs for a row-major (channel-contiguous) B operand
//   warps 14..21  builders: W (K-major, no swizzle; hi and lo) from walk_kernel's group records (walk_kernel also writes
//                 the per-pixel selection records itself).  W and the union's ids are double buffered: the build of half tile i + 1
//                 overlaps the feature streaming, MMAs and epilogue of half tile i.
// Work unit = (half tile, 256-channel half): two 256-column accumulators in TMEM, so the MMAs of unit i+1 overlap
// the epilogue of unit i.  A half tile whose union exceeds 64 columns is processed in rounds of 64 columns.
#include <cuda.h>

#include "qr_blend.cuh"

namespace qr {

constexpr int kEpiWarps = 4;
constexpr int kConvWarps = 8;                             // one union row of every stage each
constexpr int kBuildWarps = 8;                            // two pixel groups of the half tile each
constexpr int kMmaWarp = kEpiWarps;                       // warp 4
constexpr int kLoadWarp = kEpiWarps + 1;                  // warp 5
constexpr int kFirstConv = kEpiWarps + 2;                 // warps 6..13
constexpr int kFirstBuild = kFirstConv + kConvWarps;      // warps 14..21
constexpr int kMmaThreads = (kFirstBuild + kBuildWarps) * 32;
constexpr int kBuildThreads = kBuildWarps * 32;
constexpr int kGroupsPerBuild = 16 / kBuildWarps;         // pixel groups of the half tile per builder warp
constexpr int kWCols = 64;                                // union columns per round
constexpr int kUnitN = 256;                               // channels per work unit
constexpr int kStageRows = 8;                             // union rows per stage = one tf32 K step
constexpr int kStages = 2;
constexpr int kRawStages = 8;
constexpr int kRawRow = kUnitN * 4;                       // 1 KB: one feature row half
constexpr int kRawBytes = kStageRows * kRawRow;           // 8 KB per raw stage
constexpr int kWBytes = 128 * kWCols * 4;                 // 32 KB per W buffer (hi, lo)
constexpr int kStageHalf = kStageRows * kUnitN * 4;       // 8 KB (hi or lo)
constexpr int kStageBytes = 2 * kStageHalf;

struct MmaSmem {
    static constexpr int w = 0;                                           // [2 buffers][hi, lo]
    static constexpr int stages = 4 * kWBytes;
    static constexpr int raw = stages + kStages * kStageBytes;
    static constexpr int uid = raw + kRawStages * kRawBytes;              // int32[2 buffers][kWCols]
    static constexpr int bars = uid + 2 * kWCols * 4;                     // uint64[...]
    static constexpr int n_bars = 2 * kStages + 2 * kRawStages + 4 + 4;
    static constexpr int tmem = bars + n_bars * 8;
    static constexpr int total = tmem + 16;
};

__device__ __forceinline__ uint32_t s_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void bar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(s_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void bar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred P1;\n\tWAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
        "@P1 bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}"
        ::"r"(s_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(s_u32(bar)) : "memory");
}
__device__ __forceinline__ void bar_arrive_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(s_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_row(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(s_u32(dst)), "l"(src), "r"(bytes), "r"(s_u32(bar)) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar)     // arrives when every MMA issued so far by this thread is done
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(s_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
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

// byte offset of W[m][c] in the K-major, non-swizzled canonical layout: core matrix = 8 pixels x 4 columns (128 B);
// column chunks 128 B apart (LBO), 8-pixel groups 2 KB apart (SBO)
__device__ __forceinline__ uint32_t w_off(int m, int c)
{
    return (uint32_t)((m >> 3) * (kWCols / 4 * 128) + (c >> 2) * 128 + (m & 7) * 16 + (c & 3) * 4);
}

// rounds / K steps of a half tile: both the producers and the MMA thread derive them from the union size
__device__ __forceinline__ int rounds_of(int U) { return U <= kWCols ? 1 : (U + kWCols - 1) / kWCols; }
__device__ __forceinline__ int cols_of(int U, int r) { return max(0, min(kWCols, U - r * kWCols)); }
__device__ __forceinline__ int ksteps_of(int ncols) { return max(1, (ncols + kStageRows - 1) / kStageRows); }

__global__ void __launch_bounds__(kMmaThreads, 1) blend_mma_kernel(const BlendParams p)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char* stage_base = smem + MmaSmem::stages;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + MmaSmem::bars);
    uint64_t* full = bars;                       // [kStages] converters -> MMA (8 warp arrivals)
    uint64_t* empty = bars + kStages;            // [kStages] MMA -> converters (tcgen05.commit)
    uint64_t* raw_full = bars + 2 * kStages;     // [kRawStages] loader (TMA complete_tx) -> converters
    uint64_t* raw_empty = raw_full + kRawStages; // [kRawStages] converters -> loader (8 warp arrivals)
    uint64_t* w_ready = raw_empty + kRawStages;  // [2] builders -> MMA, loader: W instance i lives in buffer i & 1
    uint64_t* w_free = w_ready + 2;              // [2] MMA -> builders (tcgen05.commit)
    uint64_t* tmem_full = w_free + 2;            // [2] MMA -> epilogue (tcgen05.commit)
    uint64_t* tmem_empty = tmem_full + 2;        // [2] epilogue -> MMA (4 warp arrivals)
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + MmaSmem::tmem);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int D = p.D;
    const int nunits = D / kUnitN;
    const int num_half = p.num_tiles * 2;

    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) { bar_init(&full[s], kConvWarps); bar_init(&empty[s], 1); }
        for (int s = 0; s < kRawStages; ++s) { bar_init(&raw_full[s], 1); bar_init(&raw_empty[s], kConvWarps); }
        for (int b = 0; b < 2; ++b) {
            bar_init(&w_ready[b], 1); bar_init(&w_free[b], 1);
            bar_init(&tmem_full[b], 1); bar_init(&tmem_empty[b], kEpiWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(s_u32(tmem_slot)), "r"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    auto half_origin = [&](int ht, int& x0, int& y0) {
        const int tile = ht >> 1;
        x0 = (tile % p.cam.tiles_x) * kTile;
        y0 = (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8;
    };

    if (warp < kEpiWarps) {
        // ================================================= epilogue =================================================
        // thread = pixel m = 32 warp + lane of the half tile (row-major 16 x 8): TMEM lane m, 256 columns = channels.
        // 32 channels at a time: tcgen05.ld -> scale -> four 256-bit st.global (a lane's 32 channels are 128
        // contiguous bytes of the map, and every store instruction writes 32 whole sectors).  The first version
        // staged the tile in shared memory for a TMA tensor store; with two staging tiles per warp the epilogue
        // warps spent their time in cp.async.bulk.wait_group.read and became the critical path (profiles/README.md).
        int unit = 0;
        auto ld32 = [&](uint32_t taddr, uint32_t (&r)[32]) {
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
                         : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                           "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
                           "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
                           "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                         : "r"(taddr));
        };
        for (int ht = blockIdx.x; ht < num_half; ht += gridDim.x) {
            int x0, y0;
            half_origin(ht, x0, y0);
            if (y0 >= p.cam.height) continue;
            const int m = warp * 32 + lane;
            const int x = x0 + (m & 15), y = y0 + (m >> 4);
            const bool valid = x < p.cam.width && y < p.cam.height;
            const int64_t pix = (int64_t)y * p.cam.width + x;
            for (int c = 0; c < nunits; ++c, ++unit) {
                const int buf = unit & 1;
                bar_wait(&tmem_full[buf], (unit >> 1) & 1);
                tc_fence_after();
                const uint32_t t0 = tmem_base + ((uint32_t)(warp * 32) << 16) + (uint32_t)(buf * kUnitN);
                float* orow = p.out_map + pix * D + c * kUnitN;
                auto emit = [&](const uint32_t (&r)[32], int chunk) {
                    if (!valid) return;
                    float* dst = orow + chunk * 32;
#pragma unroll
                    for (int jj = 0; jj < 4; ++jj)
                        asm volatile("st.global.L1::no_allocate.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                                     ::"l"(dst + 8 * jj),
                                       "r"(r[8 * jj]), "r"(r[8 * jj + 1]), "r"(r[8 * jj + 2]), "r"(r[8 * jj + 3]),
                                       "r"(r[8 * jj + 4]), "r"(r[8 * jj + 5]), "r"(r[8 * jj + 6]), "r"(r[8 * jj + 7])
                                     : "memory");
                };
                uint32_t ra[32], rb[32];
                ld32(t0, ra);
#pragma unroll 1
                for (int ch = 0; ch < kUnitN / 32; ch += 2) {
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    ld32(t0 + (ch + 1) * 32, rb);
                    emit(ra, ch);
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    if (ch + 2 < kUnitN / 32) ld32(t0 + (ch + 2) * 32, ra);
                    else {                              // every tcgen05.ld of this accumulator has completed
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) bar_arrive(&tmem_empty[buf]);
                    }
                    emit(rb, ch + 1);
                }
            }
        }
    } else if (warp == kMmaWarp) {
        // ================================================= MMA issuer ===============================================
        // The whole warp runs the loop in uniform control flow (descriptors stay in uniform registers); one elected
        // lane issues the tcgen05 instructions.
        // M = 128, N = 256, fp32 accumulate, A and B tf32, A K-major, B MN-major
        const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | (1u << 16) | ((uint32_t)(kUnitN >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
        const uint32_t w0 = s_u32(smem + MmaSmem::w), st0 = s_u32(stage_base);
        int unit = 0, wb = 0, wcur = 0, st = 0;            // wb: W instances seen so far; wcur: the one in use
        for (int ht = blockIdx.x; ht < num_half; ht += gridDim.x) {
            int x0, y0;
            half_origin(ht, x0, y0);
            if (y0 >= p.cam.height) continue;
            const int U = __ldg(p.sl.hdr + (size_t)ht * kHdrWords + 4);
            const int rounds = rounds_of(U);
            for (int c = 0; c < nunits; ++c, ++unit) {
                const int buf = unit & 1;
                bar_wait(&tmem_empty[buf], ((unit >> 1) & 1) ^ 1);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + (uint32_t)(buf * kUnitN);
                for (int r = 0; r < rounds; ++r) {
                    if (c == 0 || rounds > 1) { wcur = wb++; bar_wait(&w_ready[wcur & 1], (wcur >> 1) & 1); }
                    const uint32_t a_hi = w0 + (uint32_t)(wcur & 1) * 2 * kWBytes, a_lo = a_hi + kWBytes;
                    const int nk = ksteps_of(cols_of(U, r));
                    for (int j = 0; j < nk; ++j, ++st) {
                        const int s = st % kStages;
                        bar_wait(&full[s], (st / kStages) & 1);
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
                        if (elect_one()) umma_commit(&w_free[wcur & 1]);
                        __syncwarp();
                    }
                }
                if (elect_one()) umma_commit(&tmem_full[buf]);
                __syncwarp();
            }
        }
    } else if (warp == kLoadWarp) {
        // ================================================= loader ===================================================
        // lane k < 8 copies union row 8 j + k of every stage: 1 KB (256 channels) per bulk copy, kRawStages ahead
        unsigned char* raw_base = smem + MmaSmem::raw;
        // (the union's ids come from the walk's lists in global memory: the loader never waits for a W build)
        int st = 0;
        for (int ht = blockIdx.x; ht < num_half; ht += gridDim.x) {
            int x0, y0;
            half_origin(ht, x0, y0);
            if (y0 >= p.cam.height) continue;
            const int U = __ldg(p.sl.hdr + (size_t)ht * kHdrWords + 4);
            const int rounds = rounds_of(U);
            for (int c = 0; c < nunits; ++c) {
                for (int r = 0; r < rounds; ++r) {
                    const int ncols = cols_of(U, r);
                    const int nk = ksteps_of(ncols);
                    for (int j = 0; j < nk; ++j, ++st) {
                        const int s = st % kRawStages;
                        bar_wait(&raw_empty[s], ((st / kRawStages) & 1) ^ 1);
                        const int rows = max(0, min(kStageRows, ncols - j * kStageRows));
                        if (lane == 0) {
                            if (rows > 0) bar_arrive_tx(&raw_full[s], (uint32_t)rows * kRawRow);
                            else bar_arrive(&raw_full[s]);
                        }
                        __syncwarp();
                        if (lane < rows) {
                            const int32_t id = __ldg(p.sl.uid + (size_t)ht * p.sl.ucap + r * kWCols + j * kStageRows + lane);
                            tma_row(raw_base + s * kRawBytes + lane * kRawRow,
                                    static_cast<const float*>(p.features) + (int64_t)id * D + c * kUnitN, kRawRow, &raw_full[s]);
                        }
                    }
                }
            }
        }
    } else if (warp < kFirstBuild) {
        // ================================================= converters ===============================================
        // warp pw splits union row pw of every stage: ld.shared of the raw row -> hi / lo -> st.shared in the MN-major
        // SWIZZLE_128B_BASE32B layout.  They only need the union sizes, never W, so they run ahead of the builders.
        const int pw = warp - kFirstConv;                 // 0..7
        const unsigned char* raw_base = smem + MmaSmem::raw;
        // byte offset of this lane's 16 bytes inside a stage half: channels 4 lane .. 4 lane + 3 (+128)
        const uint32_t lane_off = (uint32_t)((lane >> 3) * 1024 + (pw >> 2) * 512 + (pw & 3) * 128 +
                                             ((((lane & 7) >> 1) ^ (pw & 3)) * 32) + (lane & 1) * 16);
        int st = 0;
        for (int ht = blockIdx.x; ht < num_half; ht += gridDim.x) {
            int x0, y0;
            half_origin(ht, x0, y0);
            if (y0 >= p.cam.height) continue;
            const int U = __ldg(p.sl.hdr + (size_t)ht * kHdrWords + 4);
            const int rounds = rounds_of(U);
            for (int c = 0; c < nunits; ++c) {
                for (int r = 0; r < rounds; ++r) {
                    const int ncols = cols_of(U, r);
                    const int nk = ksteps_of(ncols);
                    for (int j = 0; j < nk; ++j, ++st) {
                        const int sr = st % kRawStages;
                        bar_wait(&raw_full[sr], (st / kRawStages) & 1);
                        float4 a0 = make_float4(0.f, 0.f, 0.f, 0.f), a1 = a0;
                        if (j * kStageRows + pw < ncols) {
                            const unsigned char* rr = raw_base + sr * kRawBytes + pw * kRawRow + lane * 16;
                            a0 = *reinterpret_cast<const float4*>(rr);
                            a1 = *reinterpret_cast<const float4*>(rr + 512);
                        }
                        const float4 h0 = make_float4(tf32_hi(a0.x), tf32_hi(a0.y), tf32_hi(a0.z), tf32_hi(a0.w));
                        const float4 h1 = make_float4(tf32_hi(a1.x), tf32_hi(a1.y), tf32_hi(a1.z), tf32_hi(a1.w));
                        const float4 l0 = make_float4(__fsub_rn(a0.x, h0.x), __fsub_rn(a0.y, h0.y), __fsub_rn(a0.z, h0.z), __fsub_rn(a0.w, h0.w));
                        const float4 l1 = make_float4(__fsub_rn(a1.x, h1.x), __fsub_rn(a1.y, h1.y), __fsub_rn(a1.z, h1.z), __fsub_rn(a1.w, h1.w));
                        __syncwarp();
                        if (lane == 0) bar_arrive(&raw_empty[sr]);          // the raw row is in registers
                        const int s = st % kStages;
                        bar_wait(&empty[s], ((st / kStages) & 1) ^ 1);
                        unsigned char* hi = stage_base + s * kStageBytes + lane_off;
                        unsigned char* lo = hi + kStageHalf;
                        *reinterpret_cast<float4*>(hi) = h0;
                        *reinterpret_cast<float4*>(hi + 4 * 1024) = h1;
                        *reinterpret_cast<float4*>(lo) = l0;
                        *reinterpret_cast<float4*>(lo + 4 * 1024) = l1;
                        fence_async_smem();
                        __syncwarp();
                        if (lane == 0) bar_arrive(&full[s]);
                    }
                }
            }
        }
    } else {
        // ================================================= builders =================================================
        // W (K-major, no swizzle; hi and lo) from the half tile's entry lists (qr_sel.cuh): thread = entry, one coalesced
        // 8-byte load each, issued before the wait on the buffer they go to; clear, scatter, publish.  W instances are
        // built one ahead of the MMAs, alternating between two buffers: the build of half tile i + 1 overlaps the
        // feature streaming, MMAs and epilogue of half tile i.
        const int ptid = tid - kFirstBuild * 32;          // 0..255
        auto prod_sync = [&]() { asm volatile("bar.sync 1, %0;" ::"n"(kBuildThreads) : "memory"); };
        constexpr int kEntRegs = 4;                       // entries a builder thread holds in flight
        int wb = 0;
        for (int ht = blockIdx.x; ht < num_half; ht += gridDim.x) {
            int x0, y0;
            half_origin(ht, x0, y0);
            if (y0 >= p.cam.height) continue;
            const int4 nq = __ldg(reinterpret_cast<const int4*>(p.sl.hdr + (size_t)ht * kHdrWords));
            const int U = __ldg(p.sl.hdr + (size_t)ht * kHdrWords + 4);
            const int e1 = nq.x, e2 = e1 + nq.y, e3 = e2 + nq.z, total = e3 + nq.w;
            const uint2* ent = p.sl.ent + (size_t)ht * kSelLists * p.sl.qcap;
            auto ent_at = [&](int f) -> uint2 {            // flat index over the four lists
                const int q = (f >= e1) + (f >= e2) + (f >= e3);
                const int b = q == 0 ? 0 : (q == 1 ? e1 : (q == 2 ? e2 : e3));
                return __ldg(ent + (size_t)q * p.sl.qcap + (f - b));
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
                        const int wcur = wb++;                     // this W instance; it lives in buffer wcur & 1
                        bar_wait(&w_free[wcur & 1], ((wcur >> 1) & 1) ^ 1);        // the MMAs that read the buffer have retired
                        unsigned char* wbuf = smem + MmaSmem::w + (wcur & 1) * 2 * kWBytes;
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
                        if (ptid == 0) bar_arrive(&w_ready[wcur & 1]);
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

int launch_blend_mma(const BlendParams& p, cudaStream_t st)
{
    static int sms = 0;
    if (sms == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
            sms = 148;
    }
    const unsigned grid = (unsigned)min(sms, p.num_tiles * 2);
    QR_CUDA_OK(cudaFuncSetAttribute(blend_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, MmaSmem::total));
    blend_mma_kernel<<<grid, kMmaThreads, MmaSmem::total, st>>>(p);
    QR_LAUNCH_OK("blend_mma_kernel");
    return QR_OK;
}

}  // namespace qr
